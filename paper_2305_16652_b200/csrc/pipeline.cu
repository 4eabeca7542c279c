// The whole per-batch hot path behind one call (Figure 11): key compute
// kernel -> ray sort kernel -> trace kernel, for the three orderings the bench compares
// (NoSort, TwoPoint, hierarchy cut code), plus the host-buffer form of the same call and the
// ANC diagnostic (Table 7).  All scratch lives in the hcc_pipeline handle, so
// nothing is allocated per batch.
#include <string.h>

#include "common.cuh"

struct hcc_pipeline {
    uint64_t n_max;
    uint32_t container_bits_max;
    bool host_staging;
    void *d_keys;
    uint32_t *d_perm[2];   // one per batch of a pair call (single calls use the first)
    uint32_t calls;        // calls made
    cudaStream_t last_stream;
    bool timing;           // record the per-stage events (hcc_pipeline_set_timing)
    void *d_ws;
    uint64_t ws_bytes;
    // hcc_reorder_trace_pair: the second batch's keys and sort run on a stream of the pipeline's own, in scratch of their own
    void *d_keys2, *d_ws2;
    cudaStream_t side;
    cudaEvent_t ev_fork, ev_join;
    float *d_rays;      // host-buffer form only
    void *d_hits;       // host-buffer form only
    cudaEvent_t ev[6];  // h2d start, encode start, sort start, trace start, trace end, d2h end
    bool timed, timed_host, host_pending;
    uint32_t sort_skip_bits;   // low key bits the sort leaves unordered (hcc_sort_range)
};

namespace hcc {

// ANC: number of distinct codes among the 32 rays of each warp, in traced
// order.  One warp per group of 32 consecutive ranks; out[0] += distinct codes, out[1] += warps.
template <typename KeyT>
__global__ void k_anc(const KeyT *__restrict__ keys, const uint32_t *__restrict__ perm, uint32_t n,
                      unsigned long long *out) {
    const uint32_t j = blockIdx.x * blockDim.x + threadIdx.x;
    const bool valid = j < n;
    const uint32_t active = __ballot_sync(0xFFFFFFFFu, valid);
    if (!valid) return;
    const KeyT k = keys[perm ? perm[j] : j];
    const uint32_t peers = __match_any_sync(active, k);
    const bool leader = (__ffs(peers) - 1) == (int)(threadIdx.x & 31u);
    const uint32_t distinct = __popc(__ballot_sync(active, leader));
    if ((threadIdx.x & 31u) == (uint32_t)(__ffs(active) - 1)) {
        atomicAdd(&out[0], (unsigned long long)distinct);
        atomicAdd(&out[1], 1ull);
    }
}

}  // namespace hcc

using namespace hcc;

extern "C" int32_t hcc_pipeline_destroy(hcc_pipeline *p) {
    if (!p) return HCC_OK;
    cudaFree(p->d_keys);
    cudaFree(p->d_perm[0]);
    cudaFree(p->d_perm[1]);
    cudaFree(p->d_ws);
    cudaFree(p->d_keys2);
    cudaFree(p->d_ws2);
    if (p->side) cudaStreamDestroy(p->side);
    if (p->ev_fork) cudaEventDestroy(p->ev_fork);
    if (p->ev_join) cudaEventDestroy(p->ev_join);
    cudaFree(p->d_rays);
    cudaFree(p->d_hits);
    for (int i = 0; i < 6; ++i)
        if (p->ev[i]) cudaEventDestroy(p->ev[i]);
    delete p;
    return HCC_OK;
}

extern "C" int32_t hcc_pipeline_create(uint64_t n_max, uint32_t container_bits_max, uint32_t flags,
                                       hcc_pipeline **out) {
    HCC_REQUIRE(out, HCC_ERR_INVALID_ARG, "hcc_pipeline_create: NULL out");
    HCC_REQUIRE((flags & ~(HCC_PIPELINE_HOST_STAGING | HCC_PIPELINE_PAIR)) == 0, HCC_ERR_INVALID_ARG, "hcc_pipeline_create: unknown flags %u", flags);
    *out = nullptr;
    HCC_REQUIRE(n_max >= 1 && n_max < (1ull << 30), HCC_ERR_INVALID_ARG, "hcc_pipeline_create: n_max must be in 1..2^30-1");
    HCC_REQUIRE(container_bits_max == 32 || container_bits_max == 64, HCC_ERR_INVALID_ARG,
                "hcc_pipeline_create: container_bits_max must be 32 or 64");
    hcc_pipeline *p = new hcc_pipeline();
    memset(p, 0, sizeof *p);
    p->n_max = n_max;
    p->container_bits_max = container_bits_max;
    p->host_staging = (flags & HCC_PIPELINE_HOST_STAGING) != 0;
    const bool pair = (flags & HCC_PIPELINE_PAIR) != 0;
    int32_t rc = hcc_sort_workspace_bytes(n_max, container_bits_max, &p->ws_bytes);
    if (rc != HCC_OK) { delete p; return rc; }
    cudaError_t e = cudaMalloc(&p->d_keys, (size_t)(container_bits_max / 8) * n_max);
    if (e == cudaSuccess) e = cudaMalloc((void **)&p->d_perm[0], sizeof(uint32_t) * n_max);
    if (e == cudaSuccess) e = cudaMalloc((void **)&p->d_perm[1], sizeof(uint32_t) * n_max);
    if (e == cudaSuccess) e = cudaMalloc(&p->d_ws, p->ws_bytes);
    if (e == cudaSuccess && p->host_staging) e = cudaMalloc((void **)&p->d_rays, 32 * n_max);
    if (e == cudaSuccess && p->host_staging) e = cudaMalloc(&p->d_hits, 16 * n_max);
    // hcc_reorder_trace_pair: the second batch's keys and sort workspace, the side stream and its fork / join events
    if (e == cudaSuccess && pair) e = cudaMalloc(&p->d_keys2, (size_t)(container_bits_max / 8) * n_max);
    if (e == cudaSuccess && pair) e = cudaMalloc(&p->d_ws2, p->ws_bytes);
    if (e == cudaSuccess && pair) e = cudaEventCreateWithFlags(&p->ev_fork, cudaEventDisableTiming);
    if (e == cudaSuccess && pair) e = cudaEventCreateWithFlags(&p->ev_join, cudaEventDisableTiming);
    if (e == cudaSuccess && pair) e = cudaStreamCreateWithFlags(&p->side, cudaStreamNonBlocking);
    for (int i = 0; i < 6 && e == cudaSuccess; ++i) e = cudaEventCreate(&p->ev[i]);
    if (e != cudaSuccess) {
        set_error("hcc_pipeline_create: %s", cudaGetErrorString(e));
        hcc_pipeline_destroy(p);
        return e == cudaErrorMemoryAllocation ? HCC_ERR_OUT_OF_MEMORY : HCC_ERR_CUDA;
    }
    *out = p;
    return HCC_OK;
}

extern "C" int32_t hcc_pipeline_set_sort_skip_bits(hcc_pipeline *p, uint32_t bits) {
    HCC_REQUIRE(p, HCC_ERR_INVALID_ARG, "hcc_pipeline_set_sort_skip_bits: NULL pipeline");
    HCC_REQUIRE(bits <= 64, HCC_ERR_INVALID_ARG, "hcc_pipeline_set_sort_skip_bits: bits > 64");
    p->sort_skip_bits = bits;
    return HCC_OK;
}

extern "C" int32_t hcc_pipeline_set_timing(hcc_pipeline *p, uint32_t enable) {
    HCC_REQUIRE(p, HCC_ERR_INVALID_ARG, "hcc_pipeline_set_timing: NULL pipeline");
    p->timing = enable != 0;
    return HCC_OK;
}

constexpr uint64_t HCC_PAIR_SIDE_MAX_RAYS = 1ull << 23;   // hcc_reorder_trace_pair: key + sort kernels of the two batches side by side up to here

struct BatchPlan {
    uint32_t container, bits_used;
};

static int32_t plan_batch(const hcc_pipeline *p, const hcc_cut *cut, int32_t order, uint32_t key_bits, uint64_t n, int32_t mode,
                          BatchPlan *out) {
    HCC_REQUIRE(order == HCC_ORDER_NOSORT || order == HCC_ORDER_TWOPOINT || order == HCC_ORDER_HCC, HCC_ERR_INVALID_ARG,
                "hcc_reorder_trace: unknown order %d", order);
    HCC_REQUIRE(n <= p->n_max, HCC_ERR_INVALID_ARG, "hcc_reorder_trace: n exceeds the pipeline's n_max");
    HCC_REQUIRE(mode == HCC_TRACE_CLOSEST || mode == HCC_TRACE_ANY, HCC_ERR_INVALID_ARG, "hcc_reorder_trace: unknown mode %d", mode);
    out->container = 32; out->bits_used = 0;
    if (order == HCC_ORDER_HCC) {
        HCC_REQUIRE(cut && cut->valid, HCC_ERR_INVALID_ARG, "hcc_reorder_trace: order HCC needs a selected cut");
        out->container = cut->container_bits;
        out->bits_used = cut->dev.bits_used;
    } else if (order == HCC_ORDER_TWOPOINT) {
        out->container = key_bits <= 32 ? 32u : 64u;
        out->bits_used = 6u * (key_bits / 6u);
    }
    HCC_REQUIRE(out->container <= p->container_bits_max, HCC_ERR_INVALID_ARG, "hcc_reorder_trace: 64-bit keys in a 32-bit pipeline");
    return HCC_OK;
}

// Key kernel -> sort kernels of one batch on stream s, as a chain of dependent launches whose first kernel is a plain
// launch; *slot receives the batch's trace work counter, zeroed by a kernel of this chain.  `events`: per-stage events.
static int32_t run_keys_sort(hcc_pipeline *p, const hcc_bvh *bvh, const hcc_cut *cut, int32_t order, uint32_t key_bits,
                             const BatchPlan &pl, const float *rays_dev, uint64_t n, void *keys, void *ws, uint32_t *perm,
                             cudaStream_t s, bool events, uint32_t **slot) {
    int32_t rc = HCC_OK;
    *slot = nullptr;
    if (events) HCC_CUDA_TRY(cudaEventRecord(p->ev[1], s));
    if (order == HCC_ORDER_HCC) rc = encode_launch(rays_dev, n, cut, keys, s, LK_FIRST);
    else if (order == HCC_ORDER_TWOPOINT) rc = encode_twopoint_launch(rays_dev, n, bvh->scene_lo, bvh->scene_hi, key_bits, keys, s, LK_FIRST);
    if (rc != HCC_OK) return rc;
    if (events) HCC_CUDA_TRY(cudaEventRecord(p->ev[2], s));
    if (n != 0) {
        *slot = trace_take_slot(bvh);
        if (order != HCC_ORDER_NOSORT) {
            const uint32_t lo = p->sort_skip_bits < pl.bits_used ? p->sort_skip_bits : pl.bits_used;
            rc = sort_launch(keys, n, pl.container, lo, pl.bits_used, perm, ws, p->ws_bytes, s, *slot, LK_CHAIN);
        } else {
            rc = trace_arm(*slot, s);
        }
        if (rc != HCC_OK) return rc;
    }
    if (events) HCC_CUDA_TRY(cudaEventRecord(p->ev[3], s));
    return HCC_OK;
}

extern "C" int32_t hcc_reorder_trace(hcc_pipeline *p, const hcc_bvh *bvh, const hcc_cut *cut, int32_t order,
                                     uint32_t key_bits, const float *rays_dev, uint64_t n, int32_t mode,
                                     void *hits_dev, uint32_t *perm_out_dev, void *stream) {
    HCC_REQUIRE(p && bvh, HCC_ERR_INVALID_ARG, "hcc_reorder_trace: NULL handle");
    cudaStream_t s = (cudaStream_t)stream;
    p->timed = false;
    p->host_pending = false;     // hcc_pipeline_synchronize waits for THIS call now (the host form sets it again afterwards)
    BatchPlan pl;
    int32_t rc = plan_batch(p, cut, order, key_bits, n, mode, &pl);
    if (rc != HCC_OK) return rc;
    uint32_t *perm = perm_out_dev ? perm_out_dev : p->d_perm[0], *slot = nullptr;
    rc = run_keys_sort(p, bvh, cut, order, key_bits, pl, rays_dev, n, p->d_keys, p->d_ws, perm, s, p->timing, &slot);
    if (rc != HCC_OK) return rc;
    // the trace kernel: a chained launch behind the kernel that zeroed its counter
    rc = trace_launch("hcc_reorder_trace", bvh, rays_dev, n, order == HCC_ORDER_NOSORT ? nullptr : perm, mode, hits_dev, nullptr, s,
                      slot, LK_CHAIN);
    if (rc != HCC_OK) return rc;
    if (p->timing) HCC_CUDA_TRY(cudaEventRecord(p->ev[4], s));
    p->timed = p->timing;
    p->timed_host = false;
    p->last_stream = s;
    p->calls += 1u;
    return HCC_OK;
}

// Both batches of one bounce in one call (PAPER.md:245-247 runs the three kernels per batch; a renderer has the diffuse
// and the shadow batch of a bounce at the same time).  Schedule:
//   stream s    : keys + sort of batch a  --+--> trace a --> trace b (dependent launch that does NOT wait for trace a)
//   side stream : keys + sort of batch b  --+   (forked from s and joined back into it by events)
// The two sorts are chains of small latency-bound kernels that fill each other's gaps; the traversal kernel of batch b
// becomes resident CTA by CTA as that of batch a runs out (its last rays leave most SMs idle), because its inputs - the
// permutation and the zeroed work counter - were complete before trace a was launched.  The two batches use scratch of
// their own (keys, sort workspace, permutation, counter, hits).  The first kernel of the NEXT call on s is a plain launch,
// ordered after both traces; the side stream is touched again only behind an event recorded on s after them.
extern "C" int32_t hcc_reorder_trace_pair(hcc_pipeline *p, const hcc_bvh *bvh, const hcc_cut *cut, int32_t order, uint32_t key_bits,
                                          const float *rays_a_dev, uint64_t n_a, int32_t mode_a, void *hits_a_dev,
                                          const float *rays_b_dev, uint64_t n_b, int32_t mode_b, void *hits_b_dev, void *stream) {
    HCC_REQUIRE(p && bvh, HCC_ERR_INVALID_ARG, "hcc_reorder_trace_pair: NULL handle");
    cudaStream_t s = (cudaStream_t)stream;
    p->timed = false;
    p->host_pending = false;
    BatchPlan pa, pb;
    int32_t rc = plan_batch(p, cut, order, key_bits, n_a, mode_a, &pa);
    if (rc == HCC_OK) rc = plan_batch(p, cut, order, key_bits, n_b, mode_b, &pb);
    if (rc != HCC_OK) return rc;
    HCC_REQUIRE(p->side, HCC_ERR_INVALID_ARG, "hcc_reorder_trace_pair: pipeline created without HCC_PIPELINE_PAIR");
    uint32_t *slot_a = nullptr, *slot_b = nullptr;
    // side by side only while the key and sort kernels are latency-bound (a few million rays): large batches fill the
    // machine on their own and two sorts at once only get in each other's way (config 3: +1-12 % when run side by side)
    if (n_a + n_b <= HCC_PAIR_SIDE_MAX_RAYS) {
        HCC_CUDA_TRY(cudaEventRecord(p->ev_fork, s));
        HCC_CUDA_TRY(cudaStreamWaitEvent(p->side, p->ev_fork, 0));
        rc = run_keys_sort(p, bvh, cut, order, key_bits, pb, rays_b_dev, n_b, p->d_keys2, p->d_ws2, p->d_perm[1], p->side, false, &slot_b);
        if (rc == HCC_OK) rc = run_keys_sort(p, bvh, cut, order, key_bits, pa, rays_a_dev, n_a, p->d_keys, p->d_ws, p->d_perm[0], s, false, &slot_a);
        // join even after an error, so the side stream never runs ahead of the caller's stream unnoticed
        cudaError_t e = cudaEventRecord(p->ev_join, p->side);
        if (e == cudaSuccess) e = cudaStreamWaitEvent(s, p->ev_join, 0);
        if (rc != HCC_OK) return rc;
        HCC_CUDA_TRY(e);
    } else {
        rc = run_keys_sort(p, bvh, cut, order, key_bits, pa, rays_a_dev, n_a, p->d_keys, p->d_ws, p->d_perm[0], s, false, &slot_a);
        if (rc == HCC_OK) rc = run_keys_sort(p, bvh, cut, order, key_bits, pb, rays_b_dev, n_b, p->d_keys2, p->d_ws2, p->d_perm[1], s, false, &slot_b);
        if (rc != HCC_OK) return rc;
    }
    const bool sorted = order != HCC_ORDER_NOSORT;
    rc = trace_launch("hcc_reorder_trace_pair", bvh, rays_a_dev, n_a, sorted ? p->d_perm[0] : nullptr, mode_a, hits_a_dev, nullptr, s,
                      slot_a, LK_FIRST);
    if (rc != HCC_OK) return rc;
    rc = trace_launch("hcc_reorder_trace_pair", bvh, rays_b_dev, n_b, sorted ? p->d_perm[1] : nullptr, mode_b, hits_b_dev, nullptr, s,
                      slot_b, n_a ? LK_OVERLAP : LK_FIRST);
    if (rc != HCC_OK) return rc;
    p->timed_host = false;
    p->last_stream = s;
    p->calls += 1u;
    return HCC_OK;
}

extern "C" int32_t hcc_reorder_trace_host_async(hcc_pipeline *p, const hcc_bvh *bvh, const hcc_cut *cut, int32_t order,
                                                uint32_t key_bits, const float *rays_host, uint64_t n, int32_t mode,
                                                void *hits_host, void *stream) {
    HCC_REQUIRE(p && p->host_staging, HCC_ERR_INVALID_ARG, "hcc_reorder_trace_host: pipeline created without host staging");
    HCC_REQUIRE(n <= p->n_max, HCC_ERR_INVALID_ARG, "hcc_reorder_trace_host: n exceeds the pipeline's n_max");
    HCC_REQUIRE(mode == HCC_TRACE_CLOSEST || mode == HCC_TRACE_ANY, HCC_ERR_INVALID_ARG, "hcc_reorder_trace_host: unknown mode %d", mode);
    if (n == 0) return HCC_OK;
    HCC_REQUIRE(rays_host && hits_host, HCC_ERR_INVALID_ARG, "hcc_reorder_trace_host: NULL argument");
    cudaStream_t s = (cudaStream_t)stream;
    if (p->timing) HCC_CUDA_TRY(cudaEventRecord(p->ev[0], s));
    HCC_CUDA_TRY(cudaMemcpyAsync(p->d_rays, rays_host, 32 * n, cudaMemcpyHostToDevice, s));

    int32_t rc = hcc_reorder_trace(p, bvh, cut, order, key_bits, p->d_rays, n, mode, p->d_hits, nullptr, stream);
    if (rc != HCC_OK) return rc;
    HCC_CUDA_TRY(cudaMemcpyAsync(hits_host, p->d_hits, (mode == HCC_TRACE_CLOSEST ? 16 : 1) * n, cudaMemcpyDeviceToHost, s));
    HCC_CUDA_TRY(cudaEventRecord(p->ev[5], s));
    p->timed_host = true;
    p->host_pending = true;
    return HCC_OK;
}

extern "C" int32_t hcc_pipeline_synchronize(hcc_pipeline *p) {
    HCC_REQUIRE(p, HCC_ERR_INVALID_ARG, "hcc_pipeline_synchronize: NULL pipeline");
    if (p->host_pending) {
        HCC_CUDA_TRY(cudaEventSynchronize(p->ev[5]));
        p->host_pending = false;
    } else if (p->timed) {
        HCC_CUDA_TRY(cudaEventSynchronize(p->ev[4]));
    } else if (p->calls) {
        HCC_CUDA_TRY(cudaStreamSynchronize(p->last_stream));
    }
    return HCC_OK;
}

extern "C" int32_t hcc_reorder_trace_host(hcc_pipeline *p, const hcc_bvh *bvh, const hcc_cut *cut, int32_t order,
                                          uint32_t key_bits, const float *rays_host, uint64_t n, int32_t mode,
                                          void *hits_host, void *stream) {
    int32_t rc = hcc_reorder_trace_host_async(p, bvh, cut, order, key_bits, rays_host, n, mode, hits_host, stream);
    if (rc != HCC_OK || n == 0) return rc;
    HCC_CUDA_TRY(cudaStreamSynchronize((cudaStream_t)stream));
    p->host_pending = false;
    return HCC_OK;
}

extern "C" int32_t hcc_pipeline_stage_ms(hcc_pipeline *p, float ms[5]) {
    HCC_REQUIRE(p && ms, HCC_ERR_INVALID_ARG, "hcc_pipeline_stage_ms: NULL argument");
    HCC_REQUIRE(p->timed, HCC_ERR_INVALID_ARG, "hcc_pipeline_stage_ms: no timed call (hcc_pipeline_set_timing first)");
    HCC_CUDA_TRY(cudaEventSynchronize(p->ev[p->timed_host ? 5 : 4]));
    for (int i = 0; i < 3; ++i) HCC_CUDA_TRY(cudaEventElapsedTime(&ms[i], p->ev[1 + i], p->ev[2 + i]));
    ms[3] = ms[4] = 0.0f;
    if (p->timed_host) {
        HCC_CUDA_TRY(cudaEventElapsedTime(&ms[3], p->ev[0], p->ev[1]));
        HCC_CUDA_TRY(cudaEventElapsedTime(&ms[4], p->ev[4], p->ev[5]));
    }
    return HCC_OK;
}

extern "C" int32_t hcc_anc(const void *keys_dev, const uint32_t *perm_dev, uint64_t n, uint32_t container_bits,
                           uint64_t *out_dev, void *stream) {
    HCC_REQUIRE(container_bits == 32 || container_bits == 64, HCC_ERR_INVALID_ARG, "hcc_anc: container_bits must be 32 or 64");
    HCC_REQUIRE(out_dev && aligned(out_dev, 16), HCC_ERR_INVALID_ARG, "hcc_anc: out_dev NULL or misaligned");
    cudaStream_t s = (cudaStream_t)stream;
    HCC_CUDA_TRY(cudaMemsetAsync(out_dev, 0, 2 * sizeof(uint64_t), s));
    if (n == 0) return HCC_OK;
    HCC_REQUIRE(keys_dev, HCC_ERR_INVALID_ARG, "hcc_anc: NULL keys");
    HCC_REQUIRE(n < (1ull << 32), HCC_ERR_UNSUPPORTED, "hcc_anc: n >= 2^32");
    const uint32_t T = 256, blocks = (uint32_t)((n + T - 1) / T);
    if (container_bits == 32)
        k_anc<uint32_t><<<blocks, T, 0, s>>>((const uint32_t *)keys_dev, perm_dev, (uint32_t)n, (unsigned long long *)out_dev);
    else
        k_anc<unsigned long long><<<blocks, T, 0, s>>>((const unsigned long long *)keys_dev, perm_dev, (uint32_t)n, (unsigned long long *)out_dev);
    HCC_CUDA_TRY(cudaGetLastError());
    return HCC_OK;
}
