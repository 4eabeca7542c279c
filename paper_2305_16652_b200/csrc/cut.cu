// (a1) cut selection: Algorithm 2 / Algorithm 3 (:222-231) as a
// warp-cooperative bounded priority queue, one warp per level table, and the level-width
// rule that maps a (K, key_bits) request onto the paper's encoders (R-ML).
#include <string.h>

#include <vector>

#include "common.cuh"

namespace hcc {

#define HCC_INVALID_NODE 0xFFFFFFFFu

// Priority as one 64-bit integer: density bits (density >= 0, so the bit pattern orders like
// the value) above the complemented node index: the maximum is "highest density, then lowest
// index".  0 marks an empty queue slot (no node has index 0xFFFFFFFF).
__device__ __forceinline__ unsigned long long make_key(const float *__restrict__ had, uint32_t node) {
    return ((unsigned long long)__float_as_uint(had[node]) << 32) | (unsigned long long)(0xFFFFFFFFu - node);
}

__device__ __forceinline__ unsigned long long warp_max_u64(unsigned long long v) {
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) {
        unsigned long long x = __shfl_xor_sync(0xFFFFFFFFu, v, o);
        v = x > v ? x : v;
    }
    return v;
}

constexpr int TABLE_WARPS = 4;

// One warp builds one table = Cut(start, w, need):
//   queue <- {start}; while len(queue) < Max and queue not empty: pop the maximum;
//   a leaf, or a node with fewer than `need` leaves below it, is retired into the table and
//   Max -= 1 (Alg. 2 lines 6-8); otherwise both children are pushed (line 10);
//   finally the queue's remainder joins the table (line 11) and the table is ordered by
//   density descending.
// The queue (<= 64 slots) lives in shared memory, two slots per lane; a pop is a warp
// arg-max.  All control flow is warp-uniform.
__global__ void __launch_bounds__(TABLE_WARPS * 32)
k_build_tables(const hcc_node *__restrict__ nodes, const float *__restrict__ had,
               const uint32_t *__restrict__ leaves, const uint32_t *__restrict__ parent_entries,
               uint32_t n_tables, uint32_t w, uint32_t need, uint32_t discard, uint32_t *__restrict__ entry_node,
               uint32_t *__restrict__ table_cnt, float4 *__restrict__ boxes) {
    __shared__ unsigned long long s_q[TABLE_WARPS][64];
    __shared__ unsigned long long s_out[TABLE_WARPS][64];
    const uint32_t lane = threadIdx.x & 31u, wib = threadIdx.x >> 5;
    const uint32_t t = blockIdx.x * TABLE_WARPS + wib;
    if (t >= n_tables) return;
    unsigned long long *q = s_q[wib], *out = s_out[wib];
    uint32_t *ent = entry_node + (size_t)t * w;
    float4 *box = boxes + 2 * (size_t)t * w;

    const uint32_t start = parent_entries ? parent_entries[t] : 0u;
    uint32_t n_out = 0;
    if (start != HCC_INVALID_NODE) {
        q[lane] = 0ull;
        q[lane + 32] = 0ull;
        __syncwarp();
        if (lane == 0) q[0] = make_key(had, start);
        __syncwarp();
        uint32_t len = 1, maxq = w;
        while (len < maxq && len > 0) {
            unsigned long long k0 = q[lane], k1 = q[lane + 32];
            unsigned long long best = k1 > k0 ? k1 : k0;
            uint32_t slot = k1 > k0 ? lane + 32 : lane;
            unsigned long long gmax = warp_max_u64(best);
            uint32_t owner = __ffs(__ballot_sync(0xFFFFFFFFu, best == gmax)) - 1;
            uint32_t gslot = __shfl_sync(0xFFFFFFFFu, slot, owner);
            uint32_t node = 0xFFFFFFFFu - (uint32_t)(gmax & 0xFFFFFFFFull);
            uint32_t count = nodes[node].count, left = nodes[node].left_or_first;
            bool expandable = count == 0 && leaves[node] >= need;
            if (!expandable) {
                if (discard) {              // literal Algorithm 3: the node is dropped
                    if (lane == 0) q[gslot] = 0ull;
                    --len;
                } else {                    // Algorithm 2 lines 6-8: retired into the list
                    if (lane == 0) { out[n_out] = gmax; q[gslot] = 0ull; }
                    ++n_out; --maxq; --len;
                }
            } else {
                if (lane == 0) q[gslot] = make_key(had, left);
                __syncwarp();
                uint32_t e0 = __ballot_sync(0xFFFFFFFFu, q[lane] == 0ull);
                uint32_t e1 = __ballot_sync(0xFFFFFFFFu, q[lane + 32] == 0ull);
                uint32_t free_slot = e0 ? (uint32_t)__ffs(e0) - 1u : 32u + (uint32_t)__ffs(e1) - 1u;
                if (lane == 0) q[free_slot] = make_key(had, left + 1u);
                ++len;
            }
            __syncwarp();
        }
        // line 11: the remainder of the queue
        unsigned long long k0 = q[lane], k1 = q[lane + 32];
        uint32_t m0 = __ballot_sync(0xFFFFFFFFu, k0 != 0ull), m1 = __ballot_sync(0xFFFFFFFFu, k1 != 0ull);
        uint32_t lt = (1u << lane) - 1u;
        if (k0 != 0ull) out[n_out + __popc(m0 & lt)] = k0;
        if (k1 != 0ull) out[n_out + __popc(m0) + __popc(m1 & lt)] = k1;
        n_out += __popc(m0) + __popc(m1);
        __syncwarp();
        // order by priority: rank = number of entries that come before (keys are distinct)
        for (uint32_t e = lane; e < n_out; e += 32) {
            unsigned long long ke = out[e];
            uint32_t rank = 0;
            for (uint32_t j = 0; j < n_out; ++j) rank += out[j] > ke;
            uint32_t node = 0xFFFFFFFFu - (uint32_t)(ke & 0xFFFFFFFFull);
            hcc_node nd = nodes[node];
            ent[rank] = node;
            // entry layout for the encoder's packed arithmetic: {lo.x, lo.y | hi.x, hi.y}, {lo.z, hi.z | cnt, -}
            box[2 * rank + 0] = make_float4(nd.lo[0], nd.lo[1], nd.hi[0], nd.hi[1]);
            box[2 * rank + 1] = make_float4(nd.lo[2], nd.hi[2], rank == 0 ? __uint_as_float(n_out) : 0.0f, 0.0f);
        }
    }
    for (uint32_t j = n_out + lane; j < w; j += 32) {   // empty slots (and empty tables: cnt = 0 in slot 0)
        ent[j] = HCC_INVALID_NODE;
        box[2 * j + 0] = make_float4(0.f, 0.f, 0.f, 0.f);
        box[2 * j + 1] = make_float4(0.f, 0.f, 0.f, 0.f);
    }
    if (lane == 0) table_cnt[t] = n_out;
}

int32_t launch_build_tables(const hcc_bvh *bvh, const float *had, hcc_cut *cut, cudaStream_t s) {
    const CutDev &d = cut->dev;
    for (uint32_t l = 0; l < d.m; ++l) {
        uint32_t need = (l + 1 < d.m) ? d.w[l + 1] : 2u;
        const uint32_t *parent_entries = l == 0 ? nullptr : cut->d_entry_node + d.ent_off[l - 1];
        uint32_t blocks = (d.n_tab[l] + TABLE_WARPS - 1) / TABLE_WARPS;
        k_build_tables<<<blocks, TABLE_WARPS * 32, 0, s>>>(
            bvh->d_nodes, had, bvh->d_leaves, parent_entries, d.n_tab[l], d.w[l], need,
            (cut->flags & HCC_CUT_ALG3_DISCARD) && l + 1 < d.m ? 1u : 0u,
            cut->d_entry_node + d.ent_off[l], cut->d_table_cnt + d.tab_off[l],
            cut->d_boxes + 2 * (size_t)d.ent_off[l]);
    }
    HCC_CUDA_TRY(cudaGetLastError());
    return HCC_OK;
}

// Reading R-ML: K <= B: one level of K entries.  Otherwise the fewest levels
// m >= 2 whose power-of-two widths (exponent of K = 2^k split as evenly as possible, larger
// first) sum to <= B; if none, k is reduced.
static uint32_t level_widths(uint32_t K, uint32_t B, uint32_t *w, uint32_t *K_eff) {
    if (K <= B) { w[0] = K; *K_eff = K; return 1; }
    uint32_t k = 31u - (uint32_t)__builtin_clz(K);
    for (; k >= 1; --k) {
        for (uint32_t m = 2; m <= k && m <= HCC_MAX_LEVELS; ++m) {
            uint32_t q = k / m, r = k % m, sum = 0;
            for (uint32_t i = 0; i < m; ++i) { w[i] = 1u << (q + (i < r ? 1u : 0u)); sum += w[i]; }
            if (sum <= B) { *K_eff = 1u << k; return m; }
        }
    }
    w[0] = K < B ? K : B; *K_eff = w[0];
    return 1;
}

}  // namespace hcc

using namespace hcc;

extern "C" int32_t hcc_cut_create(uint32_t max_K, hcc_cut **out) {
    HCC_REQUIRE(out && max_K >= 1 && max_K <= (1u << 20), HCC_ERR_INVALID_ARG, "hcc_cut_create: bad argument");
    *out = nullptr;
    hcc_cut *c = new hcc_cut();
    memset(c, 0, sizeof *c);
    // entries over all levels of a hierarchy with K finest nodes: at most K + K/2 + K/4 + ... < 2K
    // (every width >= 2), plus one flat table of up to 64
    c->cap_entries = 2u * max_K + 64u;
    c->cap_tables = max_K + 64u;
    cudaError_t e = cudaMalloc((void **)&c->d_boxes, sizeof(float4) * 2 * (size_t)c->cap_entries);
    if (e == cudaSuccess) e = cudaMalloc((void **)&c->d_entry_node, sizeof(uint32_t) * (size_t)c->cap_entries);
    if (e == cudaSuccess) e = cudaMalloc((void **)&c->d_table_cnt, sizeof(uint32_t) * (size_t)c->cap_tables);
    if (e != cudaSuccess) {
        set_error("hcc_cut_create: cudaMalloc failed: %s", cudaGetErrorString(e));
        hcc_cut_destroy(c);
        return e == cudaErrorMemoryAllocation ? HCC_ERR_OUT_OF_MEMORY : HCC_ERR_CUDA;
    }
    *out = c;
    return HCC_OK;
}

extern "C" int32_t hcc_cut_destroy(hcc_cut *c) {
    if (!c) return HCC_OK;
    cudaFree(c->d_boxes);
    cudaFree(c->d_entry_node);
    cudaFree(c->d_table_cnt);
    delete c;
    return HCC_OK;
}

static bool key_bits_ok(uint32_t b) { return b == 16 || b == 24 || b == 32 || b == 48 || b == 64; }

// Lays the level tables of widths[0..m-1] out in the handle's buffers (no kernel runs).
static int32_t set_levels(hcc_cut *cut, const uint32_t *widths, uint32_t m, uint32_t key_bits) {
    HCC_REQUIRE(key_bits_ok(key_bits), HCC_ERR_INVALID_ARG, "hcc_select_cut: key_bits must be 16, 24, 32, 48 or 64");
    HCC_REQUIRE(m >= 1 && m <= HCC_MAX_LEVELS, HCC_ERR_INVALID_ARG, "hcc_select_cut: 1..%u levels", HCC_MAX_LEVELS);
    CutDev d;
    memset(&d, 0, sizeof d);
    d.m = m;
    uint64_t ent = 0, tab = 0, nt = 1, bits = 0;
    for (uint32_t l = 0; l < m; ++l) {
        HCC_REQUIRE(widths[l] >= 1 && widths[l] <= HCC_MAX_WIDTH, HCC_ERR_INVALID_ARG,
                    "hcc_select_cut: level width %u outside 1..%u", widths[l], HCC_MAX_WIDTH);
        d.w[l] = widths[l];
        d.ent_off[l] = (uint32_t)ent;
        d.tab_off[l] = (uint32_t)tab;
        d.n_tab[l] = (uint32_t)nt;
        ent += nt * widths[l];
        tab += nt;
        nt *= widths[l];
        bits += widths[l];
        HCC_REQUIRE(ent <= cut->cap_entries && tab <= cut->cap_tables, HCC_ERR_INVALID_ARG,
                    "hcc_select_cut: hierarchy larger than the handle's capacity (hcc_cut_create max_K)");
    }
    HCC_REQUIRE(bits <= key_bits, HCC_ERR_INVALID_ARG, "hcc_select_cut: widths need %llu bits > key_bits %u",
                (unsigned long long)bits, key_bits);
    d.n_entries = (uint32_t)ent;
    d.n_tables = (uint32_t)tab;
    d.bits_used = (uint32_t)bits;
    d.boxes = cut->d_boxes;
    d.entry_node = cut->d_entry_node;
    d.table_cnt = cut->d_table_cnt;
    cut->dev = d;
    cut->key_bits = key_bits;
    cut->container_bits = key_bits <= 32 ? 32u : 64u;
    cut->K_eff = (uint32_t)(nt);
    cut->flags = 0u;
    cut->valid = true;
    return HCC_OK;
}

extern "C" int32_t hcc_select_cut_levels_ex(const hcc_bvh *bvh, const float *density_dev, const uint32_t *widths,
                                            uint32_t m, uint32_t key_bits, uint32_t flags, hcc_cut *cut, void *stream) {
    HCC_REQUIRE(bvh && density_dev && widths && cut, HCC_ERR_INVALID_ARG, "hcc_select_cut: NULL argument");
    HCC_REQUIRE(aligned(density_dev, 16), HCC_ERR_BAD_ALIGNMENT, "hcc_select_cut: density_dev not 16-byte aligned");
    HCC_REQUIRE((flags & ~(uint32_t)HCC_CUT_ALG3_DISCARD) == 0u, HCC_ERR_INVALID_ARG, "hcc_select_cut: unknown flags 0x%x", flags);
    int32_t rc = set_levels(cut, widths, m, key_bits);
    if (rc != HCC_OK) return rc;
    cut->flags = flags;
    return launch_build_tables(bvh, density_dev, cut, (cudaStream_t)stream);
}

extern "C" int32_t hcc_select_cut_levels(const hcc_bvh *bvh, const float *density_dev, const uint32_t *widths,
                                         uint32_t m, uint32_t key_bits, hcc_cut *cut, void *stream) {
    return hcc_select_cut_levels_ex(bvh, density_dev, widths, m, key_bits, 0u, cut, stream);
}

// (f4) regular grid tables; the cell rule is stated in include/hcc.h
__global__ void k_build_grid(CutDev d, uint32_t level, uint32_t halvings_before, uint32_t k, float3 lo, float3 hi,
                             uint32_t *__restrict__ entry_node, uint32_t *__restrict__ table_cnt, float4 *__restrict__ boxes) {
    const uint32_t w = d.w[level];
    const uint32_t e = blockIdx.x * blockDim.x + threadIdx.x;        // entry within the level
    if (e >= d.n_tab[level] * w) return;
    const uint32_t t = e / w, j = e % w;
    const unsigned long long path = ((unsigned long long)t << k) | j;
    const uint32_t total = halvings_before + k;
    uint32_t idx[3] = {0u, 0u, 0u}, cnt[3] = {0u, 0u, 0u};
    for (uint32_t i = 0; i < total; ++i) {
        const uint32_t bit = (uint32_t)(path >> (total - 1u - i)) & 1u;
        idx[i % 3u] = (idx[i % 3u] << 1) | bit;
        cnt[i % 3u] += 1u;
    }
    const float slo[3] = {lo.x, lo.y, lo.z}, shi[3] = {hi.x, hi.y, hi.z};
    float blo[3], bhi[3];
    for (int a = 0; a < 3; ++a) {
        const float ext = shi[a] - slo[a];
        const float cells = (float)(1u << cnt[a]);
        blo[a] = slo[a] + ext * ((float)idx[a] / cells);
        bhi[a] = idx[a] + 1u == (1u << cnt[a]) ? shi[a] : slo[a] + ext * ((float)(idx[a] + 1u) / cells);
    }
    const size_t o = d.ent_off[level] + e;
    entry_node[o] = HCC_INVALID_NODE;
    boxes[2 * o + 0] = make_float4(blo[0], blo[1], bhi[0], bhi[1]);
    boxes[2 * o + 1] = make_float4(blo[2], bhi[2], j == 0 ? __uint_as_float(w) : 0.0f, 0.0f);
    if (j == 0) table_cnt[d.tab_off[level] + t] = w;
}

extern "C" int32_t hcc_select_grid(const hcc_bvh *bvh, const uint32_t *widths, uint32_t m, uint32_t key_bits,
                                   hcc_cut *cut, void *stream) {
    HCC_REQUIRE(bvh && widths && cut, HCC_ERR_INVALID_ARG, "hcc_select_grid: NULL argument");
    uint32_t halvings = 0, ks[HCC_MAX_LEVELS];
    for (uint32_t l = 0; l < m && l < HCC_MAX_LEVELS; ++l) {
        HCC_REQUIRE(widths[l] >= 2 && (widths[l] & (widths[l] - 1u)) == 0u, HCC_ERR_INVALID_ARG,
                    "hcc_select_grid: level widths must be powers of two >= 2");
        ks[l] = 31u - (uint32_t)__builtin_clz(widths[l]);
        halvings += ks[l];
    }
    HCC_REQUIRE(halvings <= 60u, HCC_ERR_UNSUPPORTED, "hcc_select_grid: more than 60 halvings");
    int32_t rc = set_levels(cut, widths, m, key_bits);
    if (rc != HCC_OK) return rc;
    cudaStream_t s = (cudaStream_t)stream;
    const float3 lo = make_float3(bvh->scene_lo[0], bvh->scene_lo[1], bvh->scene_lo[2]);
    const float3 hi = make_float3(bvh->scene_hi[0], bvh->scene_hi[1], bvh->scene_hi[2]);
    uint32_t before = 0;
    for (uint32_t l = 0; l < m; ++l) {
        const uint32_t n = cut->dev.n_tab[l] * cut->dev.w[l];
        k_build_grid<<<(n + 255u) / 256u, 256, 0, s>>>(cut->dev, l, before, ks[l], lo, hi, cut->d_entry_node, cut->d_table_cnt, cut->d_boxes);
        before += ks[l];
    }
    HCC_CUDA_TRY(cudaGetLastError());
    return HCC_OK;
}

// Boxes of all table entries as 6 floats (lo, hi) each, in entry order (tests, diagnostics).
extern "C" int32_t hcc_cut_read_boxes(const hcc_cut *cut, float *boxes_host, void *stream) {
    HCC_REQUIRE(cut && cut->valid && boxes_host, HCC_ERR_INVALID_ARG, "hcc_cut_read_boxes: bad argument");
    cudaStream_t s = (cudaStream_t)stream;
    const size_t n = cut->dev.n_entries;
    std::vector<float> raw(8 * n);
    HCC_CUDA_TRY(cudaMemcpyAsync(raw.data(), cut->d_boxes, sizeof(float) * 8 * n, cudaMemcpyDeviceToHost, s));
    HCC_CUDA_TRY(cudaStreamSynchronize(s));
    for (size_t e = 0; e < n; ++e) {
        const float *r = raw.data() + 8 * e;   // {lo.x, lo.y, hi.x, hi.y}, {lo.z, hi.z, cnt, -}
        float *o = boxes_host + 6 * e;
        o[0] = r[0]; o[1] = r[1]; o[2] = r[4]; o[3] = r[2]; o[4] = r[3]; o[5] = r[5];
    }
    return HCC_OK;
}

extern "C" int32_t hcc_select_cut(const hcc_bvh *bvh, const float *density_dev, uint32_t K, uint32_t key_bits,
                                  hcc_cut *cut, void *stream) {
    HCC_REQUIRE(K >= 1, HCC_ERR_INVALID_ARG, "hcc_select_cut: K must be >= 1");
    HCC_REQUIRE(key_bits_ok(key_bits), HCC_ERR_INVALID_ARG, "hcc_select_cut: key_bits must be 16, 24, 32, 48 or 64");
    uint32_t w[HCC_MAX_LEVELS], K_eff = 0;
    uint32_t m = level_widths(K, key_bits, w, &K_eff);
    int32_t rc = hcc_select_cut_levels(bvh, density_dev, w, m, key_bits, cut, stream);
    if (rc == HCC_OK) cut->K_eff = K_eff;
    return rc;
}

extern "C" int32_t hcc_cut_info(const hcc_cut *cut, uint32_t *m, uint32_t *widths, uint32_t *K_eff, uint32_t *bits_used,
                                uint32_t *container_bits, uint64_t *n_entries, uint64_t *n_tables) {
    HCC_REQUIRE(cut && cut->valid, HCC_ERR_INVALID_ARG, "hcc_cut_info: no selection in this handle");
    if (m) *m = cut->dev.m;
    if (widths) for (uint32_t l = 0; l < HCC_MAX_LEVELS; ++l) widths[l] = l < cut->dev.m ? cut->dev.w[l] : 0u;
    if (K_eff) *K_eff = cut->K_eff;
    if (bits_used) *bits_used = cut->dev.bits_used;
    if (container_bits) *container_bits = cut->container_bits;
    if (n_entries) *n_entries = cut->dev.n_entries;
    if (n_tables) *n_tables = cut->dev.n_tables;
    return HCC_OK;
}

extern "C" int32_t hcc_cut_read(const hcc_cut *cut, uint32_t *entry_node_host, uint32_t *table_cnt_host, void *stream) {
    HCC_REQUIRE(cut && cut->valid && entry_node_host && table_cnt_host, HCC_ERR_INVALID_ARG, "hcc_cut_read: bad argument");
    cudaStream_t s = (cudaStream_t)stream;
    HCC_CUDA_TRY(cudaMemcpyAsync(entry_node_host, cut->d_entry_node, sizeof(uint32_t) * (size_t)cut->dev.n_entries,
                                 cudaMemcpyDeviceToHost, s));
    HCC_CUDA_TRY(cudaMemcpyAsync(table_cnt_host, cut->d_table_cnt, sizeof(uint32_t) * (size_t)cut->dev.n_tables,
                                 cudaMemcpyDeviceToHost, s));
    HCC_CUDA_TRY(cudaStreamSynchronize(s));
    return HCC_OK;
}
