// (a4) trace: software BVH traversal of the (re)ordered rays — PAPER.md:247 ("the trace
// kernel fetches the rays based on these sorted indices"), :62-64.  B200 has no RT cores;
// closest-hit and any-hit are hand-written while-while traversal kernels over 32-byte child
// records (sibling pair = one aligned 64-byte fetch through the read-only path) with a
// per-thread stack.  Compiled with -fmad=false; fmaf() appears exactly where hcc.h states it.
#include "common.cuh"

namespace hcc {

constexpr int TRACE_THREADS = 128;
constexpr int STACK_SIZE = 64;

__device__ __forceinline__ float max3(float a, float b, float c) {
    float d;
    asm("max.f32 %0, %1, %2, %3;" : "=f"(d) : "f"(a), "f"(b), "f"(c));
    return d;
}
__device__ __forceinline__ float min3(float a, float b, float c) {
    float d;
    asm("min.f32 %0, %1, %2, %3;" : "=f"(d) : "f"(a), "f"(b), "f"(c));
    return d;
}

struct Ray {
    float ox, oy, oz, tmin, dx, dy, dz, tmax, ix, iy, iz;
};

// Conservative culling test on [tmin, limit]: slab distances (lo-o)*inv, (hi-o)*inv, the far
// end widened by 2 ulp so rounding can never cull a box whose triangle the predicate accepts.
// A box whose near distance equals `limit` is kept (ties in t go to the lowest prim id).
__device__ __forceinline__ bool box_hit(const Ray &r, const float4 lo, const float4 hi, float limit, float &tn) {
    float t1x = (lo.x - r.ox) * r.ix, t2x = (hi.x - r.ox) * r.ix;
    float t1y = (lo.y - r.oy) * r.iy, t2y = (hi.y - r.oy) * r.iy;
    float t1z = (lo.z - r.oz) * r.iz, t2z = (hi.z - r.oz) * r.iz;
    tn = fmaxf(max3(fminf(t1x, t2x), fminf(t1y, t2y), fminf(t1z, t2z)), r.tmin);
    float tf = min3(fmaxf(t1x, t2x), fmaxf(t1y, t2y), fmaxf(t1z, t2z)) * 1.0000002384185791015625f;
    tf = fminf(tf, limit);
    return tn <= tf;
}

// The triangle predicate of hcc.h, operation by operation.
__device__ __forceinline__ bool tri_hit(const Ray &r, const float4 v0, const float4 e1, const float4 e2,
                                        float &t, float &u, float &v) {
    float px = fmaf(r.dy, e2.z, -(r.dz * e2.y));
    float py = fmaf(r.dz, e2.x, -(r.dx * e2.z));
    float pz = fmaf(r.dx, e2.y, -(r.dy * e2.x));
    float det = fmaf(e1.x, px, fmaf(e1.y, py, e1.z * pz));
    if (det == 0.0f) return false;
    float inv = 1.0f / det;
    float sx = r.ox - v0.x, sy = r.oy - v0.y, sz = r.oz - v0.z;
    u = fmaf(sx, px, fmaf(sy, py, sz * pz)) * inv;
    if (!(u >= 0.0f)) return false;
    float qx = fmaf(sy, e1.z, -(sz * e1.y));
    float qy = fmaf(sz, e1.x, -(sx * e1.z));
    float qz = fmaf(sx, e1.y, -(sy * e1.x));
    v = fmaf(r.dx, qx, fmaf(r.dy, qy, r.dz * qz)) * inv;
    if (!(v >= 0.0f) || !(u + v <= 1.0f)) return false;
    t = fmaf(e2.x, qx, fmaf(e2.y, qy, e2.z * qz)) * inv;
    return t > r.tmin && t < r.tmax;
}

// STATS: the same traversal also counts, per ray, the sibling pairs fetched (64 bytes each) and
// the triangle records fetched (48 bytes each), summed into stats[0], stats[1]; stats[2] = rays,
// stats[3] = deepest stack seen.  Used for the "node bytes per ray" figure only, never timed.
template <bool ANY, bool STATS>
__global__ void __launch_bounds__(TRACE_THREADS)
k_trace(const float4 *__restrict__ trec, const float4 *__restrict__ ttri, const float4 *__restrict__ rays,
        const uint32_t *__restrict__ perm, uint32_t n, void *__restrict__ hits, unsigned long long *stats) {
    uint32_t n_pairs = 0, n_tris = 0, max_sp = 0;
    const uint32_t j = blockIdx.x * TRACE_THREADS + threadIdx.x;
    if (j >= n) return;
    const uint32_t rid = perm ? perm[j] : j;
    const float4 a = __ldg(rays + 2 * (size_t)rid), b = __ldg(rays + 2 * (size_t)rid + 1);
    Ray r;
    r.ox = a.x; r.oy = a.y; r.oz = a.z; r.tmin = a.w;
    r.dx = b.x; r.dy = b.y; r.dz = b.z; r.tmax = b.w;
    r.ix = 1.0f / b.x; r.iy = 1.0f / b.y; r.iz = 1.0f / b.z;

    float best_t = r.tmax, best_u = 0.0f, best_v = 0.0f;   // culling limit; the hit's t once one is found
    uint32_t best_prim = HCC_MISS_PRIM;
    bool occluded = false;

    uint32_t stack[STACK_SIZE];
    int sp = 0;
    uint32_t cur;
    {   // root = record 1
        const float4 lo = __ldg(trec + 2), hi = __ldg(trec + 3);
        float tn;
        cur = box_hit(r, lo, hi, best_t, tn) ? __float_as_uint(lo.w) : 0u;   // 0 = nothing to do
    }
    while (cur != 0u) {
        // descend through internal nodes: cur = record index of a sibling pair's left child
        while (!(cur & 0x80000000u)) {
            const float4 *p = trec + 2 * (size_t)cur;
            const float4 l_lo = __ldg(p), l_hi = __ldg(p + 1), r_lo = __ldg(p + 2), r_hi = __ldg(p + 3);
            if (STATS) ++n_pairs;
            float tn0, tn1;
            const bool h0 = box_hit(r, l_lo, l_hi, best_t, tn0);
            const bool h1 = box_hit(r, r_lo, r_hi, best_t, tn1);
            const uint32_t ref0 = __float_as_uint(l_lo.w), ref1 = __float_as_uint(r_lo.w);
            if (h0 && h1) {
                const bool swap = tn1 < tn0;
                stack[sp++] = swap ? ref0 : ref1;
                if (STATS) max_sp = max(max_sp, (uint32_t)sp);
                cur = swap ? ref1 : ref0;
            } else if (h0) {
                cur = ref0;
            } else if (h1) {
                cur = ref1;
            } else {
                cur = sp > 0 ? stack[--sp] : 0u;
                if (cur == 0u) break;
            }
        }
        if (cur == 0u) break;
        // leaf: test its triangles
        const uint32_t first = cur & 0x0FFFFFFFu, cnt = ((cur >> 28) & 7u) + 1u;
        for (uint32_t k = 0; k < cnt; ++k) {
            const float4 *tp = ttri + 3 * (size_t)(first + k);
            const float4 v0 = __ldg(tp), e1 = __ldg(tp + 1), e2 = __ldg(tp + 2);
            float t, u, v;
            if (STATS) ++n_tris;
            if (tri_hit(r, v0, e1, e2, t, u, v)) {
                if (ANY) { occluded = true; break; }
                const uint32_t prim = __float_as_uint(v0.w);
                if (t < best_t || (t == best_t && prim < best_prim)) {
                    best_t = t; best_u = u; best_v = v; best_prim = prim;
                }
            }
        }
        if (ANY && occluded) break;
        cur = sp > 0 ? stack[--sp] : 0u;
    }
    if (STATS) {
        atomicAdd(&stats[0], (unsigned long long)n_pairs);
        atomicAdd(&stats[1], (unsigned long long)n_tris);
        atomicAdd(&stats[2], 1ull);
        atomicMax(&stats[3], (unsigned long long)max_sp);
    }
    if (ANY) {
        reinterpret_cast<uint8_t *>(hits)[rid] = occluded ? 1 : 0;
    } else {
        const bool hit = best_prim != HCC_MISS_PRIM;
        reinterpret_cast<float4 *>(hits)[rid] =
            make_float4(hit ? best_t : __int_as_float(0x7f800000), __uint_as_float(best_prim), best_u, best_v);
    }
}

}  // namespace hcc

using namespace hcc;

static int32_t trace_impl(const char *who, const hcc_bvh *bvh, const float *rays_dev, uint64_t n, const uint32_t *perm_dev,
                          int32_t mode, void *hits_dev, unsigned long long *stats_dev, void *stream) {
    HCC_REQUIRE(bvh, HCC_ERR_INVALID_ARG, "%s: NULL bvh", who);
    HCC_REQUIRE(mode == HCC_TRACE_CLOSEST || mode == HCC_TRACE_ANY, HCC_ERR_INVALID_ARG, "%s: unknown mode %d", who, mode);
    if (n == 0) return HCC_OK;
    HCC_REQUIRE(rays_dev && hits_dev, HCC_ERR_INVALID_ARG, "%s: NULL argument", who);
    HCC_REQUIRE(aligned(rays_dev, 32) && aligned(hits_dev, 16) && aligned(perm_dev, 16), HCC_ERR_BAD_ALIGNMENT,
                "%s: rays need 32-byte, hits and perm 16-byte alignment", who);
    HCC_REQUIRE(n < (1ull << 32), HCC_ERR_UNSUPPORTED, "%s: n >= 2^32", who);
    cudaStream_t s = (cudaStream_t)stream;
    const uint32_t blocks = (uint32_t)((n + TRACE_THREADS - 1) / TRACE_THREADS);
    const float4 *rays = (const float4 *)rays_dev;
    if (stats_dev) {
        if (mode == HCC_TRACE_CLOSEST)
            k_trace<false, true><<<blocks, TRACE_THREADS, 0, s>>>(bvh->d_trec, bvh->d_ttri, rays, perm_dev, (uint32_t)n, hits_dev, stats_dev);
        else
            k_trace<true, true><<<blocks, TRACE_THREADS, 0, s>>>(bvh->d_trec, bvh->d_ttri, rays, perm_dev, (uint32_t)n, hits_dev, stats_dev);
    } else {
        if (mode == HCC_TRACE_CLOSEST)
            k_trace<false, false><<<blocks, TRACE_THREADS, 0, s>>>(bvh->d_trec, bvh->d_ttri, rays, perm_dev, (uint32_t)n, hits_dev, nullptr);
        else
            k_trace<true, false><<<blocks, TRACE_THREADS, 0, s>>>(bvh->d_trec, bvh->d_ttri, rays, perm_dev, (uint32_t)n, hits_dev, nullptr);
    }
    HCC_CUDA_TRY(cudaGetLastError());
    return HCC_OK;
}

extern "C" int32_t hcc_trace(const hcc_bvh *bvh, const float *rays_dev, uint64_t n, const uint32_t *perm_dev,
                             int32_t mode, void *hits_dev, void *stream) {
    return trace_impl("hcc_trace", bvh, rays_dev, n, perm_dev, mode, hits_dev, nullptr, stream);
}

extern "C" int32_t hcc_trace_stats(const hcc_bvh *bvh, const float *rays_dev, uint64_t n, const uint32_t *perm_dev,
                                   int32_t mode, void *hits_dev, uint64_t *stats_dev, void *stream) {
    HCC_REQUIRE(stats_dev && aligned(stats_dev, 16), HCC_ERR_INVALID_ARG, "hcc_trace_stats: stats_dev NULL or misaligned");
    HCC_CUDA_TRY(cudaMemsetAsync(stats_dev, 0, 4 * sizeof(uint64_t), (cudaStream_t)stream));
    return trace_impl("hcc_trace_stats", bvh, rays_dev, n, perm_dev, mode, hits_dev, (unsigned long long *)stats_dev, stream);
}
