// (a4) trace: software BVH traversal of the (re)ordered rays — PAPER.md:247 ("the trace
// kernel fetches the rays based on these sorted indices"), :62-64.  B200 has no RT cores.
//
// Design: persistent warps pull 32-ray chunks of the (sorted) order from an
// atomic counter and refill finished lanes from the same chunk, so the rays of a warp stay
// neighbours in the sorted order; each traversal step fetches ONE 32-byte record holding both
// quantised child boxes (bvh.cu) with a 256-bit load; the warp alternates between a node phase
// and a triangle phase, each running while at least half of the live lanes take part (a
// thresholded while-while loop); the stack lives in shared memory (conflict-free, 16 deep) and
// spills to local memory below that.  Compiled with -fmad=false; fmaf() appears exactly where
// hcc.h states it for the triangle predicate, which alone defines the results.
#include "common.cuh"

namespace hcc {

constexpr int TRACE_THREADS = 128;
#ifndef HCC_TRACE_BLOCKS_PER_SM       // closest hit: 8 CTAs of 128 threads per SM (64 registers)
#define HCC_TRACE_BLOCKS_PER_SM 8
#endif
#ifndef HCC_TRACE_BLOCKS_PER_SM_ANY   // any hit carries no (t, u, v, prim): 9 CTAs per SM (56 registers)
#define HCC_TRACE_BLOCKS_PER_SM_ANY 9
#endif
#ifndef HCC_TRACE_REFILL_AT
#define HCC_TRACE_REFILL_AT 8
#endif
#ifndef HCC_TRACE_CLOSEST_STEPWISE   // closest-hit triangle phase: 1 = one triangle per lane per iteration, thresholded
#define HCC_TRACE_CLOSEST_STEPWISE 0
#endif
#ifndef HCC_TRACE_TRI_DEN            // triangle phase goes on while 1/TRI_DEN of the live lanes hold a leaf
#define HCC_TRACE_TRI_DEN 4
#endif
constexpr int TRACE_BLOCKS_PER_SM = HCC_TRACE_BLOCKS_PER_SM, TRACE_BLOCKS_PER_SM_ANY = HCC_TRACE_BLOCKS_PER_SM_ANY;
constexpr int SMEM_STACK = 16;          // entries per thread in shared memory
constexpr int STACK_SIZE = 64;          // hcc_bvh_create admits depth <= 63
constexpr uint32_t CHUNK = 32;          // rays a warp takes from the counter at a time
constexpr uint32_t REFILL_AT = HCC_TRACE_REFILL_AT;   // idle lanes that trigger a refill

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

// One grid cell index (15 bits, low or high half of w, chosen by the byte selector) -> the
// float 32768 + cell, in one PRMT: bytes {0x00, cell.lo, cell.hi, 0x47}.
__device__ __forceinline__ float cell_plane(uint32_t w, uint32_t sel) {
    uint32_t d;
    asm("prmt.b32 %0, %1, %2, %3;" : "=r"(d) : "r"(w), "r"(0x47000000u), "r"(sel));
    return __uint_as_float(d);
}
constexpr uint32_t SEL_LO = 0x7104u, SEL_HI = 0x7324u, SEL_FLIP = 0x0220u;

struct Words8 { uint32_t w[8]; };
__device__ __forceinline__ Words8 ld256(const uint32_t *p) {   // LDG.E.256 through the read-only path
    Words8 r;
    asm volatile("ld.global.nc.v8.u32 {%0,%1,%2,%3,%4,%5,%6,%7}, [%8];"
                 : "=r"(r.w[0]), "=r"(r.w[1]), "=r"(r.w[2]), "=r"(r.w[3]), "=r"(r.w[4]), "=r"(r.w[5]), "=r"(r.w[6]), "=r"(r.w[7])
                 : "l"(p));
    return r;
}

// streamed once: rays and the permutation do not displace the BVH from L1
__device__ __forceinline__ float4 ld_stream4(const float4 *p) {
    float4 r;
    asm volatile("ld.global.nc.L1::no_allocate.v4.f32 {%0,%1,%2,%3}, [%4];" : "=f"(r.x), "=f"(r.y), "=f"(r.z), "=f"(r.w) : "l"(p));
    return r;
}
__device__ __forceinline__ uint32_t ld_stream(const uint32_t *p) {
    uint32_t r;
    asm volatile("ld.global.nc.L1::no_allocate.u32 %0, [%1];" : "=r"(r) : "l"(p));
    return r;
}

struct Ray {
    float ox, oy, oz, tmin, dx, dy, dz, tmax;
};

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

struct TraceScene {
    const uint32_t *qrec;
    const float4 *ttri;
    uint32_t root_ref;
    float q_lo[3], q_scale[3];
};

// ctl[0] = next ray rank (zeroed on the launch stream before every launch).
// STATS: the same traversal also counts the pair records fetched (32 bytes each) and the
// triangle records fetched (64 bytes each): stats[0], stats[1]; stats[2] = rays, stats[3] =
// deepest stack seen; stats[4] = distinct pair records summed over warp-level node steps (what
// a coherent warp saves), stats[5] = warp-level node steps, stats[6] = lanes taking part in
// them.  Used for the diagnostics only, never timed.
template <bool ANY, bool STATS>
__global__ void __launch_bounds__(TRACE_THREADS, ANY ? TRACE_BLOCKS_PER_SM_ANY : TRACE_BLOCKS_PER_SM)
k_trace(const TraceScene sc, const float4 *__restrict__ rays, const uint32_t *__restrict__ perm, uint32_t n,
        void *__restrict__ hits, uint32_t *ctl, unsigned long long *stats) {
    __shared__ uint32_t s_stack[SMEM_STACK][TRACE_THREADS];
    uint32_t l_stack[STACK_SIZE - SMEM_STACK];
    const uint32_t tid = threadIdx.x, lane = tid & 31u;
    const uint32_t lanes_below = (1u << lane) - 1u;
    unsigned long long n_pairs = 0, n_tris = 0, n_rays = 0, n_sect = 0, n_steps = 0, n_lanes = 0;
    uint32_t max_sp = 0;

    uint32_t w_next = 0, w_end = 0;      // the warp's current chunk of ranks
    bool exhausted = false, have = false;
    uint32_t cur = 0, rid = 0;           // cur: 0 = ray finished, else a record reference
    int sp = 0;
    Ray r;
    float ix = 0.f, iy = 0.f, iz = 0.f;                                 // slab planes: t = (32768 + cell) * i + c
    float cnx = 0.f, cny = 0.f, cnz = 0.f, cfx = 0.f, cfy = 0.f, cfz = 0.f;   // c of the near / far planes
    uint32_t snx = SEL_LO, sny = SEL_LO, snz = SEL_LO;                  // near-plane selectors
    float best_t = 0.f, best_u = 0.f, best_v = 0.f;                     // culling limit / the hit
    uint32_t best_prim = HCC_MISS_PRIM;

    auto push = [&](uint32_t v) {
        if (sp < SMEM_STACK) s_stack[sp][tid] = v; else l_stack[sp - SMEM_STACK] = v;
        ++sp;
        if (STATS) max_sp = max(max_sp, (uint32_t)sp);
    };
    auto pop = [&]() -> uint32_t {
        if (sp == 0) return 0u;
        --sp;
        return sp < SMEM_STACK ? s_stack[sp][tid] : l_stack[sp - SMEM_STACK];
    };

    for (;;) {
        // ---- refill idle lanes with the next ranks of the warp's chunk
        uint32_t idle = __ballot_sync(0xFFFFFFFFu, !have);
        if (!exhausted && (idle == 0xFFFFFFFFu || (uint32_t)__popc(idle) >= REFILL_AT)) {
            while (idle) {
                if (w_next == w_end) {
                    uint32_t base = 0;
                    if (lane == 0) base = atomicAdd(&ctl[0], CHUNK);
                    base = __shfl_sync(0xFFFFFFFFu, base, 0);
                    if (base >= n) { exhausted = true; break; }
                    w_next = base;
                    w_end = min(base + CHUNK, n);
                }
                const uint32_t avail = w_end - w_next;
                const uint32_t rank = __popc(idle & lanes_below);
                if (!have && rank < avail) {
                    const uint32_t j = w_next + rank;
                    rid = perm ? ld_stream(perm + j) : j;
                    const float4 a = ld_stream4(rays + 2 * (size_t)rid), b = ld_stream4(rays + 2 * (size_t)rid + 1);
                    r.ox = a.x; r.oy = a.y; r.oz = a.z; r.tmin = a.w;
                    r.dx = b.x; r.dy = b.y; r.dz = b.z; r.tmax = b.w;
                    // the ray in grid units: g(t) = go + t * (d * scale); a zero (or denormal)
                    // direction component becomes a huge finite reciprocal so that no inf - inf
                    // arises: the ray then just does not move along that axis
                    const float BIG = 1.2676506e30f;   // 2^100
                    const float gx = ((a.x - sc.q_lo[0]) * sc.q_scale[0] + HCC_GRID_OFFSET) + 32768.0f;
                    const float gy = ((a.y - sc.q_lo[1]) * sc.q_scale[1] + HCC_GRID_OFFSET) + 32768.0f;
                    const float gz = ((a.z - sc.q_lo[2]) * sc.q_scale[2] + HCC_GRID_OFFSET) + 32768.0f;
                    ix = 1.0f / (b.x * sc.q_scale[0]); iy = 1.0f / (b.y * sc.q_scale[1]); iz = 1.0f / (b.z * sc.q_scale[2]);
                    ix = ix == ix ? fminf(fmaxf(ix, -BIG), BIG) : BIG;
                    iy = iy == iy ? fminf(fmaxf(iy, -BIG), BIG) : BIG;
                    iz = iz == iz ? fminf(fmaxf(iz, -BIG), BIG) : BIG;
                    // t(plane) = plane * i - g * i.  The rounding of g, of i and of this sum moves the
                    // ray by about (|g| + 65536) * 2^-22 cells at the box, so near planes are tested
                    // HCC_TRACE_PAD times (|g| + 65536) cells earlier and far planes that much later (an
                    // origin inside the scene: 1/8 cell; a distant origin: in proportion to its distance).
                    const float px = (fabsf(gx) + 65536.0f) * HCC_TRACE_PAD, py = (fabsf(gy) + 65536.0f) * HCC_TRACE_PAD,
                                pz = (fabsf(gz) + 65536.0f) * HCC_TRACE_PAD;
                    const float ax = fabsf(ix), ay = fabsf(iy), az = fabsf(iz);
                    cnx = -fmaf(gx, ix, px * ax); cfx = -fmaf(gx, ix, -(px * ax));
                    cny = -fmaf(gy, iy, py * ay); cfy = -fmaf(gy, iy, -(py * ay));
                    cnz = -fmaf(gz, iz, pz * az); cfz = -fmaf(gz, iz, -(pz * az));
                    snx = ix >= 0.0f ? SEL_LO : SEL_HI; sny = iy >= 0.0f ? SEL_LO : SEL_HI; snz = iz >= 0.0f ? SEL_LO : SEL_HI;
                    best_t = r.tmax; best_u = 0.f; best_v = 0.f; best_prim = HCC_MISS_PRIM;
                    sp = 0;
                    cur = sc.root_ref;
                    have = true;
                    if (STATS) ++n_rays;
                }
                w_next += min((uint32_t)__popc(idle), avail);
                idle = __ballot_sync(0xFFFFFFFFu, !have);
            }
        }
        if (__ballot_sync(0xFFFFFFFFu, have) == 0u) break;

        // ---- node phase: while at least half of the live lanes want a node step
        {
            uint32_t m = __ballot_sync(0xFFFFFFFFu, cur != 0u && !(cur & HCC_REF_LEAF));
            const uint32_t live = __popc(__ballot_sync(0xFFFFFFFFu, cur != 0u));
            const uint32_t need = (live + 1u) / 2u;
            while (m != 0u && (uint32_t)__popc(m) >= need) {
                if (STATS) {
                    const bool walking = cur != 0u && !(cur & HCC_REF_LEAF);
                    const uint32_t peers = __match_any_sync(0xFFFFFFFFu, walking ? cur : (0x40000000u | lane));
                    if (walking && (peers & lanes_below) == 0u) ++n_sect;
                    if (lane == 0) { ++n_steps; n_lanes += __popc(m); }
                }
                if (cur != 0u && !(cur & HCC_REF_LEAF)) {
                    const Words8 q = ld256(sc.qrec + 8 * (size_t)(cur - 1u));
                    if (STATS) ++n_pairs;
                    const uint32_t sfx = snx ^ SEL_FLIP, sfy = sny ^ SEL_FLIP, sfz = snz ^ SEL_FLIP;
                    float tn0 = max3(fmaf(cell_plane(q.w[0], snx), ix, cnx), fmaf(cell_plane(q.w[1], sny), iy, cny), fmaf(cell_plane(q.w[2], snz), iz, cnz));
                    float tf0 = min3(fmaf(cell_plane(q.w[0], sfx), ix, cfx), fmaf(cell_plane(q.w[1], sfy), iy, cfy), fmaf(cell_plane(q.w[2], sfz), iz, cfz));
                    float tn1 = max3(fmaf(cell_plane(q.w[3], snx), ix, cnx), fmaf(cell_plane(q.w[4], sny), iy, cny), fmaf(cell_plane(q.w[5], snz), iz, cnz));
                    float tf1 = min3(fmaf(cell_plane(q.w[3], sfx), ix, cfx), fmaf(cell_plane(q.w[4], sfy), iy, cfy), fmaf(cell_plane(q.w[5], sfz), iz, cfz));
                    tn0 = fmaxf(tn0, r.tmin); tn1 = fmaxf(tn1, r.tmin);
                    tf0 = fminf(tf0, best_t); tf1 = fminf(tf1, best_t);     // a box starting AT best_t is kept
                    const bool h0 = tn0 <= tf0, h1 = tn1 <= tf1;
                    const uint32_t ref0 = q.w[6], ref1 = q.w[7];
                    if (h0 && h1) {
                        const bool swap = tn1 < tn0;
                        push(swap ? ref0 : ref1);
                        cur = swap ? ref1 : ref0;
                    } else if (h0) cur = ref0;
                    else if (h1) cur = ref1;
                    else cur = pop();
                }
                m = __ballot_sync(0xFFFFFFFFu, cur != 0u && !(cur & HCC_REF_LEAF));
            }
        }
        // ---- triangle phase
        if (ANY || HCC_TRACE_CLOSEST_STEPWISE) {
            // one triangle per lane per iteration, while a quarter of the live lanes hold a leaf
            uint32_t m = __ballot_sync(0xFFFFFFFFu, (cur & HCC_REF_LEAF) != 0u);
            const uint32_t live = __popc(__ballot_sync(0xFFFFFFFFu, cur != 0u));
            const uint32_t need = (live + HCC_TRACE_TRI_DEN - 1u) / HCC_TRACE_TRI_DEN;
            while (m != 0u && (uint32_t)__popc(m) >= need) {
                if (cur & HCC_REF_LEAF) {
                    const uint32_t first = cur & 0x0FFFFFFFu, rem = (cur >> 28) & 7u;
                    const Words8 A = ld256(reinterpret_cast<const uint32_t *>(sc.ttri + 4 * (size_t)first));
                    const float4 e2 = __ldg(sc.ttri + 4 * (size_t)first + 2);
                    if (STATS) ++n_tris;
                    const float4 v0 = make_float4(__uint_as_float(A.w[0]), __uint_as_float(A.w[1]), __uint_as_float(A.w[2]), 0.f);
                    const float4 e1 = make_float4(__uint_as_float(A.w[4]), __uint_as_float(A.w[5]), __uint_as_float(A.w[6]), 0.f);
                    float t, u, v;
                    const bool hit = tri_hit(r, v0, e1, e2, t, u, v);
                    if (ANY) {
                        if (hit) { best_prim = 0u; sp = 0; cur = 0u; }
                        else cur = rem == 0u ? pop() : (HCC_REF_LEAF | ((rem - 1u) << 28) | (first + 1u));
                    } else {
                        const uint32_t prim = A.w[3];
                        if (hit && (t < best_t || (t == best_t && prim < best_prim))) { best_t = t; best_u = u; best_v = v; best_prim = prim; }
                        cur = rem == 0u ? pop() : (HCC_REF_LEAF | ((rem - 1u) << 28) | (first + 1u));
                    }
                }
                m = __ballot_sync(0xFFFFFFFFu, (cur & HCC_REF_LEAF) != 0u);
            }
        } else if (cur & HCC_REF_LEAF) {
            const uint32_t first = cur & 0x0FFFFFFFu, cnt = ((cur >> 28) & 7u) + 1u;
            for (uint32_t k = 0; k < cnt; ++k) {
                const float4 *tp = sc.ttri + 4 * (size_t)(first + k);
                const Words8 A = ld256(reinterpret_cast<const uint32_t *>(tp));
                const float4 e2 = __ldg(tp + 2);
                if (STATS) ++n_tris;
                const float4 v0 = make_float4(__uint_as_float(A.w[0]), __uint_as_float(A.w[1]), __uint_as_float(A.w[2]), 0.f);
                const float4 e1 = make_float4(__uint_as_float(A.w[4]), __uint_as_float(A.w[5]), __uint_as_float(A.w[6]), 0.f);
                float t, u, v;
                if (tri_hit(r, v0, e1, e2, t, u, v)) {
                    const uint32_t prim = A.w[3];
                    if (t < best_t || (t == best_t && prim < best_prim)) { best_t = t; best_u = u; best_v = v; best_prim = prim; }
                }
            }
            cur = pop();
        }
        __syncwarp();
        // ---- retire finished rays
        if (have && cur == 0u) {
            if (ANY) reinterpret_cast<uint8_t *>(hits)[rid] = best_prim != HCC_MISS_PRIM ? 1 : 0;
            else {
                const bool hit = best_prim != HCC_MISS_PRIM;
                reinterpret_cast<float4 *>(hits)[rid] =
                    make_float4(hit ? best_t : __int_as_float(0x7f800000), __uint_as_float(best_prim), best_u, best_v);
            }
            have = false;
        }
    }
    if (STATS) {
        atomicAdd(&stats[0], n_pairs);
        atomicAdd(&stats[1], n_tris);
        atomicAdd(&stats[2], n_rays);
        atomicMax(&stats[3], (unsigned long long)max_sp);
        atomicAdd(&stats[4], n_sect);
        atomicAdd(&stats[5], n_steps);
        atomicAdd(&stats[6], n_lanes);
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
    // the rank counter runs up to n + 32 * (warps of the grid) before every warp has seen it exhausted
    HCC_REQUIRE(n < (1ull << 32) - (1ull << 24), HCC_ERR_UNSUPPORTED, "%s: n >= 2^32 - 2^24", who);
    cudaStream_t s = (cudaStream_t)stream;
    const uint32_t cap = (uint32_t)sm_count() * (mode == HCC_TRACE_ANY ? TRACE_BLOCKS_PER_SM_ANY : TRACE_BLOCKS_PER_SM);
    const uint32_t want = (uint32_t)((n + TRACE_THREADS - 1) / TRACE_THREADS);
    const uint32_t blocks = want < cap ? want : cap;
    TraceScene sc;
    sc.qrec = bvh->d_qrec; sc.ttri = bvh->d_ttri; sc.root_ref = bvh->root_ref;
    for (int a = 0; a < 3; ++a) { sc.q_lo[a] = bvh->q_lo[a]; sc.q_scale[a] = bvh->q_scale[a]; }
    // every launch takes the next counter slot of the ring and zeroes it on its own stream first, so
    // launches in flight on different streams never share a counter (up to HCC_TRACE_SLOTS of them)
    // and an aborted launch leaves nothing behind
    uint32_t *ctl = bvh->d_trace_ctl + 2u * (bvh->trace_calls->fetch_add(1u) % (uint32_t)HCC_TRACE_SLOTS);
    HCC_CUDA_TRY(cudaMemsetAsync(ctl, 0, 2 * sizeof(uint32_t), s));
    const float4 *rays = (const float4 *)rays_dev;
    if (stats_dev) {
        if (mode == HCC_TRACE_CLOSEST) k_trace<false, true><<<blocks, TRACE_THREADS, 0, s>>>(sc, rays, perm_dev, (uint32_t)n, hits_dev, ctl, stats_dev);
        else                           k_trace<true, true><<<blocks, TRACE_THREADS, 0, s>>>(sc, rays, perm_dev, (uint32_t)n, hits_dev, ctl, stats_dev);
    } else {
        if (mode == HCC_TRACE_CLOSEST) k_trace<false, false><<<blocks, TRACE_THREADS, 0, s>>>(sc, rays, perm_dev, (uint32_t)n, hits_dev, ctl, nullptr);
        else                           k_trace<true, false><<<blocks, TRACE_THREADS, 0, s>>>(sc, rays, perm_dev, (uint32_t)n, hits_dev, ctl, nullptr);
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
    HCC_CUDA_TRY(cudaMemsetAsync(stats_dev, 0, 8 * sizeof(uint64_t), (cudaStream_t)stream));
    return trace_impl("hcc_trace_stats", bvh, rays_dev, n, perm_dev, mode, hits_dev, (unsigned long long *)stats_dev, stream);
}
