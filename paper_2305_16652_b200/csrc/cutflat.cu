// (a1) Algorithm 2 for ANY K as a data-parallel closed form.
//
// The density of a parent is >= that of each child (all terms of Eq. 1 are >= 0 and fp32
// rounding is monotone) and ties break toward the lower index (parent index < child index),
// so the priority queue pops nodes in the global order (density desc, index asc).  Popping a
// leaf lowers MaxQueueSize and the queue length together, so the loop ends exactly after
// K-1 INTERNAL pops.  Hence: S = the K-1 first internal nodes in that order; the cut is the
// set of children of S that are not in S (the root if S is empty), ordered by (density desc,
// index asc).  Top-(K-1) selection = the library's own radix sort.
#include <string.h>

#include "common.cuh"

namespace hcc {

// keys of the internal nodes, in ascending node-index order (ids = bvh->d_internal), so the
// stable sort breaks density ties toward the lower node index.
__global__ void k_internal_keys(const float *__restrict__ had, const uint32_t *__restrict__ ids, uint32_t n_int,
                                uint32_t *__restrict__ keys, uint32_t *counter) {
    uint32_t i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i == 0) *counter = 0u;
    if (i < n_int) keys[i] = 0xFFFFFFFFu - __float_as_uint(had[ids[i]]);    // ascending key = descending density
}

__global__ void k_mark_selected(const uint32_t *__restrict__ perm, const uint32_t *__restrict__ ids, uint32_t n_sel,
                                uint8_t *__restrict__ in_s) {
    uint32_t i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i < n_sel) in_s[ids[perm[i]]] = 1;
}

// children of S that are not in S -> list (any order), as 64-bit keys (density desc, index asc)
__global__ void k_emit_frontier(const hcc_node *__restrict__ nodes, const float *__restrict__ had,
                                const uint32_t *__restrict__ perm, const uint32_t *__restrict__ ids, uint32_t n_sel,
                                const uint8_t *__restrict__ in_s, unsigned long long *__restrict__ keys64,
                                uint32_t *counter) {
    uint32_t i = blockIdx.x * blockDim.x + threadIdx.x;
    if (n_sel == 0) {
        if (i == 0) { keys64[0] = ((unsigned long long)(0xFFFFFFFFu - __float_as_uint(had[0])) << 32); *counter = 1u; }
        return;
    }
    if (i >= n_sel) return;
    const uint32_t l = nodes[ids[perm[i]]].left_or_first;
    for (uint32_t c = l; c <= l + 1u; ++c) {
        if (!in_s[c]) {
            uint32_t slot = atomicAdd(counter, 1u);
            keys64[slot] = ((unsigned long long)(0xFFFFFFFFu - __float_as_uint(had[c])) << 32) | c;
        }
    }
}

__global__ void k_copy_keys_low(const unsigned long long *__restrict__ keys64, const uint32_t *counter,
                                unsigned long long *__restrict__ sort_keys, uint32_t *__restrict__ ids_out, uint32_t cap) {
    // pad the unused tail with the maximum key so one fixed-size sort works without a host sync
    uint32_t i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= cap) return;
    uint32_t cnt = *counter;
    unsigned long long k = i < cnt ? keys64[i] : 0xFFFFFFFFFFFFFFFFull;
    sort_keys[i] = k;
    ids_out[i] = (uint32_t)(k & 0xFFFFFFFFull);
}

__global__ void k_gather_cut(const uint32_t *__restrict__ perm, const uint32_t *__restrict__ ids_in, const uint32_t *counter,
                             uint32_t *__restrict__ out, uint32_t *count_out, uint32_t cap) {
    uint32_t i = blockIdx.x * blockDim.x + threadIdx.x;
    uint32_t cnt = *counter;
    if (i == 0) *count_out = cnt;
    if (i < cap && i < cnt) out[i] = ids_in[perm[i]];
}

struct FlatLayout {
    uint64_t keys32, perm, in_s, keys64, sort64, ids_k, perm_k, counter, sort_ws, total;
    uint64_t sort_ws_bytes;
};

static int32_t flat_layout(const hcc_bvh *bvh, uint32_t K, FlatLayout *L) {
    const uint64_t n_int = bvh->n_nodes - bvh->n_leaves;
    const uint64_t cap = K;    // frontier size <= K
    uint64_t ws_a = 0, ws_b = 0;
    int32_t rc = hcc_sort_workspace_bytes(n_int ? n_int : 1, 32, &ws_a);
    if (rc != HCC_OK) return rc;
    rc = hcc_sort_workspace_bytes(cap, 64, &ws_b);
    if (rc != HCC_OK) return rc;
    uint64_t o = 0;
    auto take = [&](uint64_t bytes) { uint64_t at = o; o += round_up(bytes ? bytes : 1, 256); return at; };
    L->keys32 = take(4 * n_int);
    L->perm = take(4 * n_int);
    L->in_s = take(bvh->n_nodes);
    L->keys64 = take(8 * (cap + 2));
    L->sort64 = take(8 * cap);
    L->ids_k = take(4 * cap);
    L->perm_k = take(4 * cap);
    L->counter = take(256);
    L->sort_ws_bytes = ws_a > ws_b ? ws_a : ws_b;
    L->sort_ws = take(L->sort_ws_bytes);
    L->total = o + 256;
    return HCC_OK;
}

}  // namespace hcc

using namespace hcc;

extern "C" int32_t hcc_select_cut_flat_workspace_bytes(const hcc_bvh *bvh, uint32_t K, uint64_t *bytes) {
    HCC_REQUIRE(bvh && bytes && K >= 1, HCC_ERR_INVALID_ARG, "hcc_select_cut_flat_workspace_bytes: bad argument");
    FlatLayout L;
    int32_t rc = flat_layout(bvh, K, &L);
    if (rc != HCC_OK) return rc;
    *bytes = L.total;
    return HCC_OK;
}

extern "C" int32_t hcc_select_cut_flat(const hcc_bvh *bvh, const float *density_dev, uint32_t K, uint32_t *cut_nodes_dev,
                                       uint32_t *count_dev, void *workspace_dev, uint64_t workspace_bytes, void *stream) {
    HCC_REQUIRE(bvh && density_dev && cut_nodes_dev && count_dev && workspace_dev, HCC_ERR_INVALID_ARG,
                "hcc_select_cut_flat: NULL argument");
    HCC_REQUIRE(K >= 1 && K <= (1u << 24), HCC_ERR_INVALID_ARG, "hcc_select_cut_flat: K must be in 1..2^24");
    HCC_REQUIRE(aligned(density_dev, 16) && aligned(cut_nodes_dev, 16) && aligned(workspace_dev, 16), HCC_ERR_BAD_ALIGNMENT,
                "hcc_select_cut_flat: pointers need 16-byte alignment");
    FlatLayout L;
    int32_t rc = flat_layout(bvh, K, &L);
    if (rc != HCC_OK) return rc;
    HCC_REQUIRE(workspace_bytes >= L.total, HCC_ERR_INVALID_ARG, "hcc_select_cut_flat: workspace too small");
    cudaStream_t s = (cudaStream_t)stream;
    unsigned char *ws = reinterpret_cast<unsigned char *>(round_up(reinterpret_cast<uintptr_t>(workspace_dev), 256));
    uint32_t *keys32 = (uint32_t *)(ws + L.keys32), *perm = (uint32_t *)(ws + L.perm);
    const uint32_t *ids = bvh->d_internal;
    uint8_t *in_s = ws + L.in_s;
    unsigned long long *keys64 = (unsigned long long *)(ws + L.keys64), *sort64 = (unsigned long long *)(ws + L.sort64);
    uint32_t *ids_k = (uint32_t *)(ws + L.ids_k), *perm_k = (uint32_t *)(ws + L.perm_k), *counter = (uint32_t *)(ws + L.counter);
    void *sort_ws = ws + L.sort_ws;

    const uint32_t n_int = bvh->n_nodes - bvh->n_leaves;
    const uint32_t n_sel = (K - 1u) < n_int ? (K - 1u) : n_int;
    const uint32_t T = 256;
    HCC_CUDA_TRY(cudaMemsetAsync(in_s, 0, bvh->n_nodes, s));
    k_internal_keys<<<(n_int + T) / T, T, 0, s>>>(density_dev, ids, n_int, keys32, counter);
    if (n_sel > 0) {
        rc = hcc_sort(keys32, n_int, 32, 32, perm, sort_ws, L.sort_ws_bytes, stream);
        if (rc != HCC_OK) return rc;
        k_mark_selected<<<(n_sel + T - 1) / T, T, 0, s>>>(perm, ids, n_sel, in_s);
    }
    k_emit_frontier<<<(n_sel ? (n_sel + T - 1) / T : 1), T, 0, s>>>(bvh->d_nodes, density_dev, perm, ids, n_sel, in_s, keys64, counter);
    // order the frontier by (density desc, index asc); fixed size K with max-key padding
    k_copy_keys_low<<<(K + T - 1) / T, T, 0, s>>>(keys64, counter, sort64, ids_k, K);
    rc = hcc_sort(sort64, K, 64, 64, perm_k, sort_ws, L.sort_ws_bytes, stream);
    if (rc != HCC_OK) return rc;
    k_gather_cut<<<(K + T - 1) / T, T, 0, s>>>(perm_k, ids_k, counter, cut_nodes_dev, count_dev, K);
    HCC_CUDA_TRY(cudaGetLastError());
    return HCC_OK;
}
