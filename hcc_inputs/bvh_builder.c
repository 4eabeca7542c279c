/* Deterministic host binned-SAH BVH builder: part of the generated INPUT
 * (BASELINE.json north_star: "deterministic host binned-SAH builder (16 bins,
 * fixed tie-breaking) that is part of the generated input").
 *
 * It is the one piece of native code that both the oracle's tests and the CUDA
 * path's tests consume (through the arrays it writes).  It holds none of the
 * method's arithmetic: no density, no cut search, no ray test, no sort.
 *
 * Canonical BVH (the array both sides take):
 *   node = { float lo[3], hi[3]; uint32 left_or_first; uint32 count; }   32 bytes
 *   count == 0 : internal, children are nodes left_or_first and left_or_first+1
 *   count  > 0 : leaf, triangles prim_idx[left_or_first .. left_or_first+count)
 * Rules: binary; leaf <= max_leaf triangles; a node with more is always split;
 * bins over the bounds of the triangles' box centres, all three axes, n_bins-1
 * candidate planes each; cost = A(L)*N(L) + A(R)*N(R) in fp32 (A = half area);
 * strictly-lower cost wins, so ties keep the lower axis, then the lower plane;
 * no usable plane (coincident centres) -> split the index range in half;
 * the partition is stable.  Nodes are numbered in the order they are created
 * while scanning i = 0,1,2,... (breadth-first): parent index < child index and
 * siblings are adjacent (right = left + 1).
 */
#include <float.h>
#include <stdint.h>
#include <stdlib.h>
#include <string.h>

typedef struct {
    float lo[3];
    float hi[3];
    uint32_t left_or_first;
    uint32_t count;
} hcc_node;

#define MAX_BINS 64

static inline float fminf_(float a, float b) { return a < b ? a : b; }
static inline float fmaxf_(float a, float b) { return a > b ? a : b; }

static inline float half_area(const float lo[3], const float hi[3]) {
    float dx = hi[0] - lo[0], dy = hi[1] - lo[1], dz = hi[2] - lo[2];
    return dx * dy + dy * dz + dz * dx;
}

/* Returns 0 on success, <0 on error.  nodes_out must hold 2*n_tris entries
 * (at least 1), prim_idx_out n_tris entries, depth_out (optional) 2*n_tris. */
int hcc_build_bvh(const float *tris, uint32_t n_tris, uint32_t max_leaf, uint32_t n_bins,
                  hcc_node *nodes_out, uint32_t *prim_idx_out, uint32_t *n_nodes_out,
                  uint32_t *max_depth_out) {
    if (!tris || !nodes_out || !prim_idx_out || !n_nodes_out) return -1;
    if (n_tris == 0 || max_leaf == 0 || n_bins < 2 || n_bins > MAX_BINS) return -1;

    float *tlo = (float *)malloc(sizeof(float) * 3 * (size_t)n_tris);
    float *thi = (float *)malloc(sizeof(float) * 3 * (size_t)n_tris);
    float *cen = (float *)malloc(sizeof(float) * 3 * (size_t)n_tris);
    uint32_t *tmp = (uint32_t *)malloc(sizeof(uint32_t) * (size_t)n_tris);
    uint8_t *side = (uint8_t *)malloc((size_t)n_tris);
    uint32_t *first = (uint32_t *)malloc(sizeof(uint32_t) * 2 * (size_t)n_tris);
    uint32_t *cnt = (uint32_t *)malloc(sizeof(uint32_t) * 2 * (size_t)n_tris);
    uint32_t *depth = (uint32_t *)malloc(sizeof(uint32_t) * 2 * (size_t)n_tris);
    if (!tlo || !thi || !cen || !tmp || !side || !first || !cnt || !depth) {
        free(tlo); free(thi); free(cen); free(tmp); free(side); free(first); free(cnt); free(depth);
        return -2;
    }

    for (uint32_t t = 0; t < n_tris; ++t) {
        const float *v = tris + 9 * (size_t)t;
        for (int a = 0; a < 3; ++a) {
            float l = fminf_(v[a], fminf_(v[3 + a], v[6 + a]));
            float h = fmaxf_(v[a], fmaxf_(v[3 + a], v[6 + a]));
            tlo[3 * (size_t)t + a] = l;
            thi[3 * (size_t)t + a] = h;
            cen[3 * (size_t)t + a] = 0.5f * (l + h);
        }
        prim_idx_out[t] = t;
    }

    uint32_t n_nodes = 1, max_depth = 0;
    first[0] = 0; cnt[0] = n_tris; depth[0] = 0;

    for (uint32_t i = 0; i < n_nodes; ++i) {
        const uint32_t f = first[i], c = cnt[i];
        hcc_node *nd = &nodes_out[i];
        float lo[3] = {FLT_MAX, FLT_MAX, FLT_MAX}, hi[3] = {-FLT_MAX, -FLT_MAX, -FLT_MAX};
        float clo[3] = {FLT_MAX, FLT_MAX, FLT_MAX}, chi[3] = {-FLT_MAX, -FLT_MAX, -FLT_MAX};
        for (uint32_t k = f; k < f + c; ++k) {
            const size_t t = prim_idx_out[k];
            for (int a = 0; a < 3; ++a) {
                lo[a] = fminf_(lo[a], tlo[3 * t + a]);
                hi[a] = fmaxf_(hi[a], thi[3 * t + a]);
                clo[a] = fminf_(clo[a], cen[3 * t + a]);
                chi[a] = fmaxf_(chi[a], cen[3 * t + a]);
            }
        }
        memcpy(nd->lo, lo, sizeof lo);
        memcpy(nd->hi, hi, sizeof hi);
        if (depth[i] > max_depth) max_depth = depth[i];
        if (c <= max_leaf) {
            nd->left_or_first = f;
            nd->count = c;
            continue;
        }

        /* binned SAH over the three axes */
        float best_cost = FLT_MAX;
        int best_axis = -1;
        uint32_t best_plane = 0;
        for (int a = 0; a < 3; ++a) {
            const float ext = chi[a] - clo[a];
            if (!(ext > 0.0f)) continue;
            const float scale = (float)n_bins / ext;
            float blo[MAX_BINS][3], bhi[MAX_BINS][3];
            uint32_t bcnt[MAX_BINS];
            for (uint32_t b = 0; b < n_bins; ++b) {
                bcnt[b] = 0;
                for (int d = 0; d < 3; ++d) { blo[b][d] = FLT_MAX; bhi[b][d] = -FLT_MAX; }
            }
            for (uint32_t k = f; k < f + c; ++k) {
                const size_t t = prim_idx_out[k];
                int b = (int)((cen[3 * t + a] - clo[a]) * scale);
                if (b < 0) b = 0;
                if (b >= (int)n_bins) b = (int)n_bins - 1;
                bcnt[b]++;
                for (int d = 0; d < 3; ++d) {
                    blo[b][d] = fminf_(blo[b][d], tlo[3 * t + d]);
                    bhi[b][d] = fmaxf_(bhi[b][d], thi[3 * t + d]);
                }
            }
            /* right-to-left suffix areas, then left-to-right sweep */
            float rarea[MAX_BINS];
            uint32_t rcnt[MAX_BINS];
            float rl[3] = {FLT_MAX, FLT_MAX, FLT_MAX}, rh[3] = {-FLT_MAX, -FLT_MAX, -FLT_MAX};
            uint32_t rc = 0;
            for (int b = (int)n_bins - 1; b >= 1; --b) {
                rc += bcnt[b];
                for (int d = 0; d < 3; ++d) { rl[d] = fminf_(rl[d], blo[b][d]); rh[d] = fmaxf_(rh[d], bhi[b][d]); }
                rcnt[b] = rc;
                rarea[b] = rc ? half_area(rl, rh) : 0.0f;
            }
            float ll[3] = {FLT_MAX, FLT_MAX, FLT_MAX}, lh[3] = {-FLT_MAX, -FLT_MAX, -FLT_MAX};
            uint32_t lc = 0;
            for (uint32_t p = 0; p + 1 < n_bins; ++p) {   /* plane p: bins 0..p left */
                lc += bcnt[p];
                for (int d = 0; d < 3; ++d) { ll[d] = fminf_(ll[d], blo[p][d]); lh[d] = fmaxf_(lh[d], bhi[p][d]); }
                if (lc == 0 || rcnt[p + 1] == 0) continue;
                const float cost = half_area(ll, lh) * (float)lc + rarea[p + 1] * (float)rcnt[p + 1];
                if (cost < best_cost) { best_cost = cost; best_axis = a; best_plane = p; }
            }
        }

        uint32_t n_left = 0;
        if (best_axis >= 0) {
            const int a = best_axis;
            const float scale = (float)n_bins / (chi[a] - clo[a]);
            for (uint32_t k = f; k < f + c; ++k) {
                const size_t t = prim_idx_out[k];
                int b = (int)((cen[3 * t + a] - clo[a]) * scale);
                if (b < 0) b = 0;
                if (b >= (int)n_bins) b = (int)n_bins - 1;
                side[k] = (uint8_t)((uint32_t)b > best_plane);
                n_left += !side[k];
            }
            /* stable partition */
            uint32_t wl = 0, wr = n_left;
            for (uint32_t k = f; k < f + c; ++k) {
                if (side[k]) tmp[wr++] = prim_idx_out[k]; else tmp[wl++] = prim_idx_out[k];
            }
            memcpy(prim_idx_out + f, tmp, sizeof(uint32_t) * c);
        } else {
            n_left = c / 2;   /* coincident centres: split the range in half, order kept */
        }

        nd->left_or_first = n_nodes;
        nd->count = 0;
        first[n_nodes] = f;              cnt[n_nodes] = n_left;
        first[n_nodes + 1] = f + n_left; cnt[n_nodes + 1] = c - n_left;
        depth[n_nodes] = depth[n_nodes + 1] = depth[i] + 1;
        n_nodes += 2;
    }

    *n_nodes_out = n_nodes;
    if (max_depth_out) *max_depth_out = max_depth;
    free(tlo); free(thi); free(cen); free(tmp); free(side); free(first); free(cnt); free(depth);
    return 0;
}
