/* ORACLE — TEST INFRASTRUCTURE ONLY.
 *
 * A plain, slow, single-threaded CPU statement of what the hot path of
 * "Faster Ray Tracing through Hierarchy Cut Code" (arxiv 2305.16652; the text is
 * /root/reference/PAPER.md, cited below as PAPER.md:<line>) computes.  Only
 * tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference
 * legs may load this library.  It shares no code with paper_2305_16652_b200/
 * (the CUDA path) and neither includes the other.
 *
 * Build: gcc -O2 -std=c11 -ffp-contract=off -fno-fast-math  (oracle/build.py).
 * Every floating-point operation below is a single IEEE-754 binary32 operation,
 * rounded to nearest even; a fused multiply-add happens only where fmaf() is
 * written.  Where the paper is silent the reading taken is the one DESIGN.md
 * lists (R1..), named at the function.
 *
 * Pins (tests/test_oracle_*.py, -m "not gpu"): HAD closed forms on hand trees;
 * Alg. 2 invariants + breadth-first special case + Fig. 7 leaf rule + the
 * top-(K-1) closed form; Fig. 8 / Fig. 9 bit layout; keys vs an independent
 * fp64 slab test; Morton closed forms; numpy stable argsort; brute-force
 * all-triangle intersection.  "parity unpinned": none of the functions here; the
 * reordering *benefit* (speed-ups, ANC) is unpinned by nature.
 */
#include <math.h>
#include <stdint.h>
#include <stdlib.h>
#include <string.h>

typedef struct {
    float lo[3];
    float hi[3];
    uint32_t left_or_first; /* internal: left child (right = left+1); leaf: first slot in prim_idx */
    uint32_t count;         /* 0 = internal, else number of triangles of the leaf */
} node_t;

#define INVALID_U32 0xFFFFFFFFu

/* ------------------------------------------------------------------------- */
/* (a1) Hierarchically accumulated density — PAPER.md:185-188, Eq. 1 (:187)   */
/* ------------------------------------------------------------------------- */

/* SA: the paper does not print the formula; R1: SA = 2(dx*dy + dy*dz + dz*dx),
 * evaluated left to right in fp32. */
static float surface_area(const node_t *n) {
    float dx = n->hi[0] - n->lo[0];
    float dy = n->hi[1] - n->lo[1];
    float dz = n->hi[2] - n->lo[2];
    return 2.0f * ((dx * dy + dy * dz) + dz * dx);
}

/* Eq. 1: leaf  HAD = TC * SA;  internal  HAD = HAD_left + HAD_right + lambda * SA.
 * R2: evaluated as (HAD_l + HAD_r) + (lambda * SA).  Children have larger indices
 * than their parent (canonical BVH), so one descending scan is bottom-up. */
void oracle_had(const node_t *nodes, uint32_t n_nodes, float lambda, float *had) {
    for (uint32_t k = n_nodes; k-- > 0;) {
        const node_t *n = &nodes[k];
        float sa = surface_area(n);
        if (n->count > 0) {
            had[k] = (float)n->count * sa;
        } else {
            uint32_t l = n->left_or_first;
            had[k] = (had[l] + had[l + 1]) + (lambda * sa);
        }
    }
}

/* Number of leaves below each node (used by Alg. 3's "large enough subtree"). */
void oracle_subtree_leaves(const node_t *nodes, uint32_t n_nodes, uint32_t *leaves) {
    for (uint32_t k = n_nodes; k-- > 0;) {
        const node_t *n = &nodes[k];
        leaves[k] = n->count > 0 ? 1u : leaves[n->left_or_first] + leaves[n->left_or_first + 1];
    }
}

/* ------------------------------------------------------------------------- */
/* (a1) Algorithm 2 / Algorithm 3 (:222-231) cut search    */
/* ------------------------------------------------------------------------- */

/* Priority: higher HAD first; R3: equal HAD -> lower node index first. */
static int before(const float *had, uint32_t a, uint32_t b) {
    if (had[a] != had[b]) return had[a] > had[b];
    return a < b;
}

typedef struct { uint32_t *v; uint32_t n; } heap_t;

static void heap_push(heap_t *h, const float *had, uint32_t x) {
    uint32_t i = h->n++;
    h->v[i] = x;
    while (i > 0) {
        uint32_t p = (i - 1) / 2;
        if (!before(had, h->v[i], h->v[p])) break;
        uint32_t t = h->v[i]; h->v[i] = h->v[p]; h->v[p] = t;
        i = p;
    }
}

static uint32_t heap_pop(heap_t *h, const float *had) {
    uint32_t top = h->v[0];
    h->v[0] = h->v[--h->n];
    uint32_t i = 0;
    for (;;) {
        uint32_t l = 2 * i + 1, r = l + 1, m = i;
        if (l < h->n && before(had, h->v[l], h->v[m])) m = l;
        if (r < h->n && before(had, h->v[r], h->v[m])) m = r;
        if (m == i) break;
        uint32_t t = h->v[i]; h->v[i] = h->v[m]; h->v[m] = t;
        i = m;
    }
    return top;
}

static const float *g_sort_had; /* single-threaded oracle: a file-level comparator context */
static int cmp_cut(const void *a, const void *b) {
    uint32_t x = *(const uint32_t *)a, y = *(const uint32_t *)b;
    if (x == y) return 0;
    return before(g_sort_had, x, y) ? -1 : 1;
}

/* Cut(start, max_size, need):
 *   Algorithm 2 started at `start` instead of the root (line 3), MaxQueueSize = max_size
 *   (line 2).  Line 6 "Node is leaf" is generalised to "Node is not expandable": a leaf,
 *   or (Alg. 3 line 6, "has large enough subtree") a node with fewer than `need` leaves
 *   below it.  need = 2 is Algorithm 2 verbatim (every internal node has >= 2 leaves).
 *   R4 (flagged deviation): Alg. 3 as printed DROPS a node that is not large
 *   enough; here it is retired INTO the list exactly like Alg. 2's leaf (lines 6-8), so
 *   the result stays an antichain covering every leaf.
 *   R5: line 10 "Push the child" = push both children.  R6: the loop also stops when the
 *   queue is empty (a BVH with fewer than max_size leaves), so the result is all leaves.
 *   Output: sorted by HAD descending, ties -> lower index.
 * Returns the number of cut nodes written to out (<= max_size).
 * discard != 0 (f4, the literal Algorithm 3, "we discard the top-level
 *   node that does not have a sufficient subtree"): a popped node that is not expandable is
 *   dropped - not added to the list, MaxQueueSize unchanged (Alg. 3 has no lines 7-8).  The
 *   result may then leave leaves uncovered and may be empty. */
uint32_t oracle_cut_ex(const node_t *nodes, const float *had, const uint32_t *leaves,
                       uint32_t start, uint32_t max_size, uint32_t need, int discard, uint32_t *out) {
    if (max_size == 0) return 0;
    heap_t pq;
    pq.v = (uint32_t *)malloc(sizeof(uint32_t) * ((size_t)max_size + 2));
    pq.n = 0;
    uint32_t n_out = 0;                       /* line 1: clear CutNodeList */
    uint32_t max_queue = max_size;            /* line 2 */
    heap_push(&pq, had, start);               /* line 3 */
    while (pq.n < max_queue && pq.n > 0) {    /* line 4 (+R6) */
        uint32_t nd = heap_pop(&pq, had);     /* line 5 */
        int expandable = nodes[nd].count == 0 && leaves[nd] >= need;
        if (!expandable) {                    /* line 6 */
            if (!discard) {
                out[n_out++] = nd;            /* line 7 */
                max_queue -= 1;               /* line 8 */
            }                                 /* Alg. 3: the node is simply gone */
        } else {                              /* line 9 */
            heap_push(&pq, had, nodes[nd].left_or_first);      /* line 10 */
            heap_push(&pq, had, nodes[nd].left_or_first + 1);
        }
    }
    for (uint32_t i = 0; i < pq.n; ++i) out[n_out++] = pq.v[i];   /* line 11 */
    free(pq.v);
    g_sort_had = had;
    qsort(out, n_out, sizeof(uint32_t), cmp_cut);
    return n_out;
}

uint32_t oracle_cut(const node_t *nodes, const float *had, const uint32_t *leaves,
                    uint32_t start, uint32_t max_size, uint32_t need, uint32_t *out) {
    return oracle_cut_ex(nodes, had, leaves, start, max_size, need, 0, out);
}

/* Multi-level tables (MLHCC, generalised to m levels by reading
 * R-ML of SURVEY.md §8(c)-A / DESIGN.md):
 *   level 0 has one table  = Cut(root, w[0], need_0)
 *   level l has prod(w[0..l-1]) table slots; the table of entry e of level l-1 (slot e)
 *                          = Cut(node(e), w[l], need_l);  an empty entry has an empty table
 *   need_l = w[l+1] for l < m-1, and 2 on the last level (pure Alg. 2).
 * entry_node: concatenation over levels of n_tables[l]*w[l] node ids (INVALID_U32 = empty);
 * table_cnt:  concatenation over levels of n_tables[l] entry counts.
 * discard != 0: every level that has a level below it is built by the literal Algorithm 3
 * (oracle_cut_ex with discard); the last level is Algorithm 2 either way ("follows a
 * similar method as HCC"). */
void oracle_level_tables_ex(const node_t *nodes, const float *had, const uint32_t *leaves,
                            const uint32_t *w, uint32_t m, int discard, uint32_t *entry_node, uint32_t *table_cnt) {
    size_t ent_off = 0, tab_off = 0, prev_ent_off = 0;
    size_t n_tables = 1;
    for (uint32_t l = 0; l < m; ++l) {
        uint32_t need = (l + 1 < m) ? w[l + 1] : 2u;
        for (size_t t = 0; t < n_tables; ++t) {
            uint32_t *dst = entry_node + ent_off + t * w[l];
            for (uint32_t j = 0; j < w[l]; ++j) dst[j] = INVALID_U32;
            uint32_t start = (l == 0) ? 0u : entry_node[prev_ent_off + t];
            uint32_t c = 0;
            if (start != INVALID_U32) c = oracle_cut_ex(nodes, had, leaves, start, w[l], need, discard && l + 1 < m, dst);
            table_cnt[tab_off + t] = c;
        }
        prev_ent_off = ent_off;
        ent_off += n_tables * w[l];
        tab_off += n_tables;
        n_tables *= w[l];
    }
}

void oracle_level_tables(const node_t *nodes, const float *had, const uint32_t *leaves,
                         const uint32_t *w, uint32_t m, uint32_t *entry_node, uint32_t *table_cnt) {
    oracle_level_tables_ex(nodes, had, leaves, w, m, 0, entry_node, table_cnt);
}

/* ------------------------------------------------------------------------- */
/* (a2) Encoding — Algorithm 1, MLHCC (:208-220)           */
/* ------------------------------------------------------------------------- */

/* Alg. 1 line 5 "Compute intersection between CutNode and Ray".  R7: the slab test,
 * every operation a rounded fp32 operation:
 *   inv_a = 1/d_a;  t1 = (lo_a - o_a)*inv_a;  t2 = (hi_a - o_a)*inv_a
 *   tn = max(tmin, max_a min(t1,t2));  tf = min(tmax, min_a max(t1,t2));  hit <=> tn <= tf
 * fminf/fmaxf are IEEE minNum/maxNum (a NaN operand is dropped).  d_a = +-0 gives
 * inv = +-inf: strictly between the planes t1,t2 = -+inf (the slab does not constrain),
 * outside them both are the same infinity (miss), and exactly ON a plane one product is
 * 0*inf = NaN, dropped, and the other infinity empties the slab: a miss.  The ray's own
 * [tmin,tmax] is used (R8), so a shadow ray sets no bit of a box beyond its light sample. */
static int slab_hit(const float *ray, const float *lo, const float *hi) {
    float tn = ray[3], tf = ray[7];
    float nmax = -INFINITY, fmin_ = INFINITY;
    for (int a = 0; a < 3; ++a) {
        float inv = 1.0f / ray[4 + a];
        float t1 = (lo[a] - ray[a]) * inv;
        float t2 = (hi[a] - ray[a]) * inv;
        nmax = fmaxf(nmax, fminf(t1, t2));
        fmin_ = fminf(fmin_, fmaxf(t1, t2));
    }
    tn = fmaxf(tn, nmax);
    tf = fminf(tf, fmin_);
    return tn <= tf;
}

int oracle_slab_hit(const float *ray, const float *lo, const float *hi) { return slab_hit(ray, lo, hi); }

/* Hierarchy cut code of every ray (PAPER.md:146-153 for one level; :208, :218-220 for the
 * levels below).  Bit layout R9 (PAPER.md:192 higher HAD -> higher bit; :202 node 0 = first
 * bit; :216/:220 top field above low field): the key is right-aligned in B_used = sum(w)
 * bits; field l sits directly below field l-1; entry j (HAD-descending) of a field of
 * width w is bit (w-1-j) of that field.  The representative of a level is the first hit
 * entry in HAD order (:218); a level with no hit zeroes all lower fields. */
void oracle_encode_hcc(const float *rays, uint64_t n_rays, const node_t *nodes,
                       const uint32_t *w, uint32_t m, const uint32_t *entry_node,
                       const uint32_t *table_cnt, uint64_t *keys) {
    for (uint64_t r = 0; r < n_rays; ++r) {
        const float *ray = rays + 8 * r;
        uint64_t key = 0;
        size_t ent_off = 0, tab_off = 0, n_tables = 1, table = 0;
        int alive = 1;
        for (uint32_t l = 0; l < m; ++l) {
            uint64_t mask = 0;
            int rep = -1;
            if (alive) {
                uint32_t c = table_cnt[tab_off + table];
                const uint32_t *ent = entry_node + ent_off + table * w[l];
                for (uint32_t j = 0; j < c; ++j) {           /* Alg. 1 line 4 */
                    const node_t *cn = &nodes[ent[j]];
                    if (slab_hit(ray, cn->lo, cn->hi)) {      /* line 5 */
                        mask |= (uint64_t)1 << (w[l] - 1 - j); /* line 6 */
                        if (rep < 0) rep = (int)j;
                    }
                }
            }
            key = (key << w[l]) | mask;
            if (rep < 0) alive = 0; else table = table * w[l] + (size_t)rep;
            ent_off += n_tables * w[l];
            tab_off += n_tables;
            n_tables *= w[l];
        }
        keys[r] = key;
    }
}

/* (f4) Regular grid encoding — PAPER.md:243: "the BVH cut nodes are replaced by grids that
 * divide the space evenly".  Reading R14 (the paper gives no layout): the level tables of the
 * hierarchy cut code are kept (widths w[0..m-1], powers of two) and every table entry is a
 * cell of a regular subdivision of the scene box: a cell is named by its path of halvings,
 * halving i (counted from the root, across levels) splits axis i mod 3, bit 0 = lower half;
 * entry j of a table is the cell whose log2(w) path bits of that level are j (first halving
 * in the most significant bit).  With n_a halvings of axis a so far and cell index i_a:
 *   lo_a = scene_lo_a + (scene_hi_a - scene_lo_a) * (i_a / 2^n_a)        (three fp32 operations)
 *   hi_a = the same at i_a + 1, and exactly scene_hi_a for the last cell.
 * boxes: 6 floats (lo, hi) per entry, tables laid out like oracle_level_tables. */
void oracle_grid_tables(const float *scene_lo, const float *scene_hi, const uint32_t *w, uint32_t m, float *boxes) {
    size_t ent_off = 0, n_tables = 1;
    uint32_t halvings = 0;
    for (uint32_t l = 0; l < m; ++l) {
        uint32_t k = 0;
        while ((1u << k) < w[l]) ++k;
        for (size_t t = 0; t < n_tables; ++t) {
            for (uint32_t j = 0; j < w[l]; ++j) {
                /* path of the cell: the table's path (t, halvings bits) followed by j (k bits) */
                uint64_t path = ((uint64_t)t << k) | j;
                uint32_t total = halvings + k;
                uint32_t idx[3] = {0, 0, 0}, cnt[3] = {0, 0, 0};
                for (uint32_t i = 0; i < total; ++i) {
                    uint32_t bit = (uint32_t)(path >> (total - 1 - i)) & 1u;
                    idx[i % 3] = (idx[i % 3] << 1) | bit;
                    cnt[i % 3] += 1;
                }
                float *b = boxes + 6 * (ent_off + t * w[l] + j);
                for (int a = 0; a < 3; ++a) {
                    float ext = scene_hi[a] - scene_lo[a];
                    float cells = (float)(1u << cnt[a]);
                    b[a] = scene_lo[a] + ext * ((float)idx[a] / cells);
                    b[3 + a] = idx[a] + 1u == (1u << cnt[a]) ? scene_hi[a] : scene_lo[a] + ext * ((float)(idx[a] + 1u) / cells);
                }
            }
        }
        ent_off += n_tables * w[l];
        n_tables *= w[l];
        halvings += k;
    }
}

/* The multi-level code of oracle_encode_hcc over explicit boxes (6 floats per entry) instead of
 * BVH nodes: same levels, same bit layout R9, same representative rule. */
void oracle_encode_tables(const float *rays, uint64_t n_rays, const float *boxes, const uint32_t *w, uint32_t m,
                          const uint32_t *table_cnt, uint64_t *keys) {
    for (uint64_t r = 0; r < n_rays; ++r) {
        const float *ray = rays + 8 * r;
        uint64_t key = 0;
        size_t ent_off = 0, tab_off = 0, n_tables = 1, table = 0;
        int alive = 1;
        for (uint32_t l = 0; l < m; ++l) {
            uint64_t mask = 0;
            int rep = -1;
            if (alive) {
                uint32_t c = table_cnt[tab_off + table];
                const float *b = boxes + 6 * (ent_off + table * w[l]);
                for (uint32_t j = 0; j < c; ++j) {
                    if (slab_hit(ray, b + 6 * j, b + 6 * j + 3)) {
                        mask |= (uint64_t)1 << (w[l] - 1 - j);
                        if (rep < 0) rep = (int)j;
                    }
                }
            }
            key = (key << w[l]) | mask;
            if (rep < 0) alive = 0; else table = table * w[l] + (size_t)rep;
            ent_off += n_tables * w[l];
            tab_off += n_tables;
            n_tables *= w[l];
        }
        keys[r] = key;
    }
}

/* (f3) Prefix path code — PAPER.md:116-128 (section 4.1, Figure 5): "the prefix path code is formed
 * by setting each bit to 1 if the corresponding node intersection result is true, and 0
 * otherwise ... when the rays are forced to traverse the BVH in the same order", the traversal
 * "terminat[ed] ... after a certain number of bits have been set".  Reading R13: depth-first,
 * left child before right child, starting with the root's own test; every node popped is
 * tested (slab test R7 on the ray's [tmin, tmax]) and contributes one bit, first test in the
 * most significant of the `bits` bits; a hit internal node pushes its children, a hit leaf
 * does nothing more (no triangle tests); the walk stops after `bits` tests or when the stack
 * is empty (remaining low bits zero).  Returns -1 if the fixed stack overflowed. */
int oracle_encode_ppc(const float *rays, uint64_t n_rays, const node_t *nodes, uint32_t bits, uint64_t *keys) {
    enum { PPC_STACK = 128 };
    for (uint64_t r = 0; r < n_rays; ++r) {
        const float *ray = rays + 8 * r;
        uint32_t stack[PPC_STACK];
        int sp = 0;
        uint64_t key = 0;
        uint32_t done = 0;
        stack[sp++] = 0;
        while (sp > 0 && done < bits) {
            const node_t *nd = &nodes[stack[--sp]];
            int hit = slab_hit(ray, nd->lo, nd->hi);
            key = (key << 1) | (uint64_t)hit;
            ++done;
            if (hit && nd->count == 0) {
                if (sp + 2 > PPC_STACK) return -1;
                stack[sp++] = nd->left_or_first + 1; /* right: visited after the whole left subtree */
                stack[sp++] = nd->left_or_first;
            }
        }
        keys[r] = done < bits ? key << (bits - done) : key;
    }
    return 0;
}

/* TwoPoint (details R10): origin and the estimated termination
 * point o + (0.25*e)*d (e = largest extent of the scene box, d unit) are quantised to
 * b = floor(B/6) bits per coordinate inside the scene box and bit-interleaved in the order
 * o.x o.y o.z t.x t.y t.z from the most significant bit down; right-aligned in 6b bits. */
static uint32_t quantise(float p, float lo, float hi, uint32_t b) {
    float ext = hi - lo;
    if (!(ext > 0.0f)) return 0;
    float x = ((p - lo) / ext) * (float)(1u << b);
    if (!(x >= 0.0f)) return 0;                       /* negative or NaN */
    if (x >= (float)(1u << b)) return (1u << b) - 1u;
    return (uint32_t)x;
}

void oracle_encode_twopoint(const float *rays, uint64_t n_rays, const float *scene_lo,
                            const float *scene_hi, uint32_t key_bits, uint64_t *keys) {
    uint32_t b = key_bits / 6;
    float e = fmaxf(fmaxf(scene_hi[0] - scene_lo[0], scene_hi[1] - scene_lo[1]),
                    scene_hi[2] - scene_lo[2]);
    float len = 0.25f * e;
    for (uint64_t r = 0; r < n_rays; ++r) {
        const float *ray = rays + 8 * r;
        uint32_t q[6];
        for (int a = 0; a < 3; ++a) {
            float pt = ray[a] + len * ray[4 + a];
            q[a] = quantise(ray[a], scene_lo[a], scene_hi[a], b);
            q[3 + a] = quantise(pt, scene_lo[a], scene_hi[a], b);
        }
        uint64_t key = 0;
        for (int i = (int)b - 1; i >= 0; --i)
            for (int c = 0; c < 6; ++c) key = (key << 1) | ((q[c] >> i) & 1u);
        keys[r] = key;
    }
}

/* ------------------------------------------------------------------------- */
/* (a3) Sort — PAPER.md:196 "sorting the HCCs as natural numbers", :247        */
/* ------------------------------------------------------------------------- */

/* Stable ascending order of ray ids by key: a textbook top-down merge sort on (key, id).
 * perm[j] = id of the ray at sorted rank j; equal keys keep ascending id. */
static void merge_sort(uint64_t *k, uint32_t *v, uint64_t *tk, uint32_t *tv, size_t lo, size_t hi) {
    if (hi - lo < 2) return;
    size_t mid = lo + (hi - lo) / 2;
    merge_sort(k, v, tk, tv, lo, mid);
    merge_sort(k, v, tk, tv, mid, hi);
    size_t i = lo, j = mid, o = lo;
    while (i < mid && j < hi) {
        if (k[j] < k[i]) { tk[o] = k[j]; tv[o++] = v[j++]; }     /* strict: left wins ties */
        else             { tk[o] = k[i]; tv[o++] = v[i++]; }
    }
    while (i < mid) { tk[o] = k[i]; tv[o++] = v[i++]; }
    while (j < hi)  { tk[o] = k[j]; tv[o++] = v[j++]; }
    memcpy(k + lo, tk + lo, sizeof(uint64_t) * (hi - lo));
    memcpy(v + lo, tv + lo, sizeof(uint32_t) * (hi - lo));
}

int oracle_sort(const uint64_t *keys, uint64_t n, uint32_t *perm) {
    if (n == 0) return 0;
    uint64_t *k = (uint64_t *)malloc(sizeof(uint64_t) * n), *tk = (uint64_t *)malloc(sizeof(uint64_t) * n);
    uint32_t *tv = (uint32_t *)malloc(sizeof(uint32_t) * n);
    if (!k || !tk || !tv) { free(k); free(tk); free(tv); return -1; }
    memcpy(k, keys, sizeof(uint64_t) * n);
    for (uint64_t i = 0; i < n; ++i) perm[i] = (uint32_t)i;
    merge_sort(k, perm, tk, tv, 0, n);
    free(k); free(tk); free(tv);
    return 0;
}

/* (f1) Sort truncation — PAPER.md:428 (section 6.6.1): "skip the last few bits during encoding
 * and terminate bucket sorting early".  Reading: the order is the stable ascending order of the
 * keys with their low bit_lo bits dropped, so rays whose codes differ only in those bits keep
 * their input order.  Written out as that definition: shift, then the same stable sort. */
int oracle_sort_from_bit(const uint64_t *keys, uint64_t n, uint32_t bit_lo, uint32_t *perm) {
    uint64_t *k = (uint64_t *)malloc(sizeof(uint64_t) * (n ? n : 1));
    if (!k) return -1;
    for (uint64_t i = 0; i < n; ++i) k[i] = bit_lo >= 64 ? 0 : keys[i] >> bit_lo;
    int rc = oracle_sort(k, n, perm);
    free(k);
    return rc;
}

/* ------------------------------------------------------------------------- */
/* (a4) Trace — PAPER.md:247 (trace kernel), :62-64; definition R11            */
/* ------------------------------------------------------------------------- */

/* One fixed fp32 Moeller-Trumbore form (the paper does not give the triangle test).
 * Products-of-sums use fmaf exactly where written:
 *   cross(a,b).x = fmaf(a.y, b.z, -(a.z*b.y))   (y, z cyclic)
 *   dot(a,b)     = fmaf(a.x, b.x, fmaf(a.y, b.y, a.z*b.z))
 *   e1 = v1-v0, e2 = v2-v0, p = cross(d,e2), det = dot(e1,p); det == 0 -> miss
 *   inv = 1/det, s = o-v0, u = dot(s,p)*inv, q = cross(s,e1), v = dot(d,q)*inv,
 *   t = dot(e2,q)*inv;   hit <=> u >= 0 && v >= 0 && u+v <= 1 && tmin < t < tmax.
 * No back-face culling. */
static void cross3(const float *a, const float *b, float *c) {
    c[0] = fmaf(a[1], b[2], -(a[2] * b[1]));
    c[1] = fmaf(a[2], b[0], -(a[0] * b[2]));
    c[2] = fmaf(a[0], b[1], -(a[1] * b[0]));
}
static float dot3(const float *a, const float *b) {
    return fmaf(a[0], b[0], fmaf(a[1], b[1], a[2] * b[2]));
}

static int tri_hit(const float *ray, const float *tri, float *t_out, float *u_out, float *v_out) {
    float e1[3], e2[3], p[3], s[3], q[3];
    for (int a = 0; a < 3; ++a) { e1[a] = tri[3 + a] - tri[a]; e2[a] = tri[6 + a] - tri[a]; }
    cross3(ray + 4, e2, p);
    float det = dot3(e1, p);
    if (det == 0.0f) return 0;
    float inv = 1.0f / det;
    for (int a = 0; a < 3; ++a) s[a] = ray[a] - tri[a];
    float u = dot3(s, p) * inv;
    if (!(u >= 0.0f)) return 0;
    cross3(s, e1, q);
    float v = dot3(ray + 4, q) * inv;
    if (!(v >= 0.0f) || !(u + v <= 1.0f)) return 0;
    float t = dot3(e2, q) * inv;
    if (!(t > ray[3] && t < ray[7])) return 0;
    *t_out = t; *u_out = u; *v_out = v;
    return 1;
}

int oracle_tri_hit(const float *ray, const float *tri, float *tuv) {
    return tri_hit(ray, tri, &tuv[0], &tuv[1], &tuv[2]);
}

/* Closest hit by definition: minimum t over ALL triangles; ties in t -> lowest triangle id.
 * Miss: t = +inf, prim = INVALID_U32, u = v = 0. */
void oracle_closest_brute(const float *rays, uint64_t n_rays, const float *tris, uint32_t n_tris,
                          float *hit_t, uint32_t *hit_prim, float *hit_u, float *hit_v) {
    for (uint64_t r = 0; r < n_rays; ++r) {
        float bt = INFINITY, bu = 0.0f, bv = 0.0f;
        uint32_t bp = INVALID_U32;
        for (uint32_t k = 0; k < n_tris; ++k) {
            float t, u, v;
            if (tri_hit(rays + 8 * r, tris + 9 * (size_t)k, &t, &u, &v) && t < bt) {
                bt = t; bu = u; bv = v; bp = k;
            }
        }
        hit_t[r] = bt; hit_prim[r] = bp; hit_u[r] = bu; hit_v[r] = bv;
    }
}

/* Any hit by definition: does any triangle satisfy the predicate. */
void oracle_any_brute(const float *rays, uint64_t n_rays, const float *tris, uint32_t n_tris,
                      uint8_t *occluded) {
    for (uint64_t r = 0; r < n_rays; ++r) {
        uint8_t occ = 0;
        for (uint32_t k = 0; k < n_tris && !occ; ++k) {
            float t, u, v;
            occ = (uint8_t)tri_hit(rays + 8 * r, tris + 9 * (size_t)k, &t, &u, &v);
        }
        occluded[r] = occ;
    }
}

/* The same two results through the BVH (what makes config-2-sized batches affordable).
 * Culling must never skip a triangle the predicate accepts, so the box test is the slab
 * test of R7 on [tmin, t_best] with the far end widened by 2 ulp (R12); a box whose
 * near distance EQUALS t_best is still visited so that equal-t ties resolve to the
 * lowest triangle id exactly as in the brute-force definition. */
static int slab_cull(const float *ray, const float *inv, const node_t *n, float t_best) {
    float nmax = -INFINITY, fmin_ = INFINITY;
    for (int a = 0; a < 3; ++a) {
        float t1 = (n->lo[a] - ray[a]) * inv[a];
        float t2 = (n->hi[a] - ray[a]) * inv[a];
        nmax = fmaxf(nmax, fminf(t1, t2));
        fmin_ = fminf(fmin_, fmaxf(t1, t2));
    }
    float tn = fmaxf(ray[3], nmax);
    float tf = fminf(t_best, fmin_ * 1.0000002384185791015625f);
    return !(tn <= tf);   /* 1 = culled */
}

#define STACK_MAX 256

/* stats (optional, may be NULL): [0] += nodes whose box was tested, [1] += triangles tested */
/* Both return 0, or -1 if the fixed stack overflowed (deeper than STACK_MAX: results invalid). */
int oracle_closest_bvh(const float *rays, uint64_t n_rays, const node_t *nodes,
                       const uint32_t *prim_idx, const float *tris,
                       float *hit_t, uint32_t *hit_prim, float *hit_u, float *hit_v,
                       uint64_t *stats) {
    uint64_t n_box = 0, n_tri = 0;
    int overflow = 0;
    for (uint64_t r = 0; r < n_rays; ++r) {
        const float *ray = rays + 8 * r;
        float inv[3] = {1.0f / ray[4], 1.0f / ray[5], 1.0f / ray[6]};
        float bt = INFINITY, bu = 0.0f, bv = 0.0f, lim = ray[7];
        uint32_t bp = INVALID_U32;
        uint32_t stack[STACK_MAX];
        int sp = 0;
        stack[sp++] = 0;
        while (sp > 0) {
            const node_t *n = &nodes[stack[--sp]];
            ++n_box;
            if (slab_cull(ray, inv, n, bp == INVALID_U32 ? lim : bt)) continue;
            if (n->count > 0) {
                for (uint32_t k = 0; k < n->count; ++k) {
                    uint32_t id = prim_idx[n->left_or_first + k];
                    float t, u, v;
                    ++n_tri;
                    if (tri_hit(ray, tris + 9 * (size_t)id, &t, &u, &v) &&
                        (t < bt || (t == bt && id < bp))) {
                        bt = t; bu = u; bv = v; bp = id;
                    }
                }
            } else if (sp + 2 <= STACK_MAX) {
                stack[sp++] = n->left_or_first + 1;
                stack[sp++] = n->left_or_first;
            } else {
                overflow = 1;
            }
        }
        hit_t[r] = bt; hit_prim[r] = bp; hit_u[r] = bu; hit_v[r] = bv;
    }
    if (stats) { stats[0] += n_box; stats[1] += n_tri; }
    return overflow ? -1 : 0;
}

int oracle_any_bvh(const float *rays, uint64_t n_rays, const node_t *nodes,
                   const uint32_t *prim_idx, const float *tris, uint8_t *occluded,
                   uint64_t *stats) {
    uint64_t n_box = 0, n_tri = 0;
    int overflow = 0;
    for (uint64_t r = 0; r < n_rays; ++r) {
        const float *ray = rays + 8 * r;
        float inv[3] = {1.0f / ray[4], 1.0f / ray[5], 1.0f / ray[6]};
        uint8_t occ = 0;
        uint32_t stack[STACK_MAX];
        int sp = 0;
        stack[sp++] = 0;
        while (sp > 0 && !occ) {
            const node_t *n = &nodes[stack[--sp]];
            ++n_box;
            if (slab_cull(ray, inv, n, ray[7])) continue;
            if (n->count > 0) {
                for (uint32_t k = 0; k < n->count && !occ; ++k) {
                    uint32_t id = prim_idx[n->left_or_first + k];
                    float t, u, v;
                    ++n_tri;
                    occ = (uint8_t)tri_hit(ray, tris + 9 * (size_t)id, &t, &u, &v);
                }
            } else if (sp + 2 <= STACK_MAX) {
                stack[sp++] = n->left_or_first + 1;
                stack[sp++] = n->left_or_first;
            } else {
                overflow = 1;
            }
        }
        occluded[r] = occ;
    }
    if (stats) { stats[0] += n_box; stats[1] += n_tri; }
    return overflow ? -1 : 0;
}
