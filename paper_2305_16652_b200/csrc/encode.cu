// (a2) key computation: hierarchy cut code (Algorithm 1), its multi-level
// compressed form (:204-237) and the TwoPoint comparison key (:92, :241).
// Compiled with -fmad=false: the slab test is the IEEE operation sequence hcc.h states.
#include "common.cuh"

namespace hcc {

__device__ __forceinline__ float max3(float a, float b, float c) {
    float d;
    asm("max.f32 %0, %1, %2, %3;" : "=f"(d) : "f"(a), "f"(b), "f"(c));   // FMNMX3, NaN operands dropped
    return d;
}
__device__ __forceinline__ float min3(float a, float b, float c) {
    float d;
    asm("min.f32 %0, %1, %2, %3;" : "=f"(d) : "f"(a), "f"(b), "f"(c));
    return d;
}

// One 32-byte ray as a single streaming 256-bit load (LDG.E.256, no L1 allocation): a warp reads
// 1024 contiguous bytes per instruction.
__device__ __forceinline__ void ld_ray(const float4 *p, float4 &a, float4 &b) {
    asm volatile("ld.global.nc.L1::no_allocate.v8.f32 {%0,%1,%2,%3,%4,%5,%6,%7}, [%8];"
                 : "=f"(a.x), "=f"(a.y), "=f"(a.z), "=f"(a.w), "=f"(b.x), "=f"(b.y), "=f"(b.z), "=f"(b.w) : "l"(p));
}

// Packed fp32 pairs (sm_100a add/mul.f32x2): two IEEE operations per issue slot, same rounding as
// the scalar forms, so the slab arithmetic below is still the operation sequence hcc.h states.
typedef unsigned long long f32x2;
__device__ __forceinline__ f32x2 pack2(float lo, float hi) {
    f32x2 r;
    asm("mov.b64 %0, {%1, %2};" : "=l"(r) : "f"(lo), "f"(hi));
    return r;
}
__device__ __forceinline__ void unpack2(f32x2 v, float &lo, float &hi) {
    asm("mov.b64 {%0, %1}, %2;" : "=f"(lo), "=f"(hi) : "l"(v));
}
__device__ __forceinline__ f32x2 sub2(f32x2 a, f32x2 b) {
    f32x2 d;
    asm("sub.rn.f32x2 %0, %1, %2;" : "=l"(d) : "l"(a), "l"(b));
    return d;
}
__device__ __forceinline__ f32x2 mul2(f32x2 a, f32x2 b) {
    f32x2 d;
    asm("mul.rn.f32x2 %0, %1, %2;" : "=l"(d) : "l"(a), "l"(b));
    return d;
}

struct RayEnc {
    f32x2 oxy, ozz, ixy, izz;   // (o.x, o.y), (o.z, o.z), (1/d.x, 1/d.y), (1/d.z, 1/d.z)
    float tmin, tmax;
};

// Cut box entry in memory (cut.cu): A = {lo.x, lo.y | hi.x, hi.y}, B = {lo.z, hi.z | cnt, -}.
// Alg. 1 line 5: t1 = (lo - o) * inv, t2 = (hi - o) * inv per axis (subtract, round, multiply,
// round), tn = max(tmin, max_a min(t1,t2)), tf = min(tmax, min_a max(t1,t2)), hit <=> tn <= tf.
// min/max drop NaN operands, so the reduction order does not matter.
__device__ __forceinline__ bool slab_hit(const RayEnc &r, const ulonglong2 A, const f32x2 Bz) {
    float t1x, t1y, t2x, t2y, t1z, t2z;
    unpack2(mul2(sub2(A.x, r.oxy), r.ixy), t1x, t1y);
    unpack2(mul2(sub2(A.y, r.oxy), r.ixy), t2x, t2y);
    unpack2(mul2(sub2(Bz, r.ozz), r.izz), t1z, t2z);
    float tn = fmaxf(max3(fminf(t1x, t2x), fminf(t1y, t2y), fminf(t1z, t2z)), r.tmin);
    float tf = fminf(min3(fmaxf(t1x, t2x), fmaxf(t1y, t2y), fmaxf(t1z, t2z)), r.tmax);
    return tn <= tf;
}

__device__ __forceinline__ ulonglong2 ldg_u2(const ulonglong2 *p) {
    ulonglong2 r;
    asm volatile("ld.global.nc.v2.u64 {%0,%1}, [%2];" : "=l"(r.x), "=l"(r.y) : "l"(p));
    return r;
}

// Mask of one table over entries [j0, j1): entry j -> bit (j1-1-j) of the result (<= 32 entries).
template <bool SMEM>
__device__ __forceinline__ uint32_t table_mask(const RayEnc &r, const ulonglong2 *__restrict__ box, uint32_t j0, uint32_t j1) {
    uint32_t mask = 0;
#pragma unroll 4
    for (uint32_t j = j0; j < j1; ++j) {
        ulonglong2 A, B;
        if (SMEM) { A = box[2 * j]; B = box[2 * j + 1]; }
        else      { A = ldg_u2(box + 2 * j); B = ldg_u2(box + 2 * j + 1); }
        mask = (mask << 1) | (slab_hit(r, A, B.x) ? 1u : 0u);
    }
    return mask;
}

// ---- staged (shared-memory) tables: the oriented form of the same test.
// A staged entry is three 16-byte units, one per axis a: {lo_a, hi_a, -hi_a, -lo_a}.  A ray that moves in +a reads the pair at
// byte 0 and keeps its origin; one that moves in -a reads the pair at byte 8 and negates its origin and reciprocal.  Either
// way (pair - o') * |inv| is (t_near, t_far) of that axis in this order, BIT FOR BIT the t1 / t2 of slab_hit (negating both
// operands of a subtraction or one of a multiplication negates the rounded result), so the six per-axis min/max disappear:
// tn = max(tmin, max_a t_near), tf = min(tmax, min_a t_far).  Only a ray with a zero (or NaN) direction component can
// tell the two forms apart (0 * inf = NaN is dropped by min/max but would be SELECTED here): those rays take slab_hit.
struct RayOri {
    f32x2 ox, oy, oz, ix, iy, iz;   // (o'_a, o'_a), (|inv_a|, |inv_a|)
    uint32_t bx, by, bz;            // byte offset of the axis pair inside an entry: 16 * a + (8 if the ray moves in -a)
};

__device__ __forceinline__ f32x2 lds_pair(uint32_t addr) {
    f32x2 v;
    asm volatile("ld.shared.b64 %0, [%1];" : "=l"(v) : "r"(addr));
    return v;
}

// Mask of one staged table over entries [j0, j1): entry j -> bit (j1-1-j).  ent = shared-window address of entry 0.
__device__ __forceinline__ uint32_t staged_mask(const RayOri &q, float tmin, float tmax, uint32_t ent, uint32_t j0, uint32_t j1) {
    uint32_t mask = 0;
#pragma unroll 4
    for (uint32_t j = j0; j < j1; ++j) {
        const uint32_t e = ent + 48u * j;
        float nx, fx, ny, fy, nz, fz;
        unpack2(mul2(sub2(lds_pair(e + q.bx), q.ox), q.ix), nx, fx);
        unpack2(mul2(sub2(lds_pair(e + q.by), q.oy), q.iy), ny, fy);
        unpack2(mul2(sub2(lds_pair(e + q.bz), q.oz), q.iz), nz, fz);
        const float tn = fmaxf(max3(nx, ny, nz), tmin);
        const float tf = fminf(min3(fx, fy, fz), tmax);
        mask = (mask << 1) | (tn <= tf ? 1u : 0u);
    }
    return mask;
}

// The same table for a ray with a zero or NaN direction component: slab_hit on the (lo, hi) pairs of the staged entries.
__device__ __forceinline__ uint32_t staged_mask_generic(const RayEnc &r, uint32_t ent, uint32_t j0, uint32_t j1) {
    uint32_t mask = 0;
    for (uint32_t j = j0; j < j1; ++j) {
        const uint32_t e = ent + 48u * j;
        float lx, hx, ly, hy, lz, hz;
        unpack2(lds_pair(e), lx, hx);
        unpack2(lds_pair(e + 16u), ly, hy);
        unpack2(lds_pair(e + 32u), lz, hz);
        ulonglong2 A;
        A.x = pack2(lx, ly); A.y = pack2(hx, hy);
        mask = (mask << 1) | (slab_hit(r, A, pack2(lz, hz)) ? 1u : 0u);
    }
    return mask;
}

constexpr int ENC_THREADS = 256;
// The HCC encoder runs one CTA of 1,024 threads per SM (64 registers, 32 warps): with the oriented tables below the kernel
// keeps two forms of the ray in registers, and 64 registers without spills beat more warps at 40 (two CTAs of 768: +14 %).
#ifndef HCC_ENC_STAGE_BYTES           // whole levels of the cut are staged in shared memory, top down, while they fit this
#define HCC_ENC_STAGE_BYTES (160 * 1024)
#endif
constexpr int ENC_HCC_THREADS = 1024;

// Alg. 1: line 1 "copy cut nodes from global memory into shared memory" (the first
// smem_entries entries = whole levels), line 2 grid-stride "while have ray", lines 4-6 per
// level.  One ray per thread per iteration; a 32-byte ray is read with ONE 256-bit load (ld.global.nc.v8.f32).
template <typename KeyT>
__global__ void __launch_bounds__(ENC_HCC_THREADS, 1)
k_encode_hcc(const float4 *__restrict__ rays, uint64_t n, const CutDev cut, uint32_t smem_entries,
             KeyT *__restrict__ keys, int wait) {
    extern __shared__ ulonglong2 s_box[];
    const ulonglong2 *g_box = reinterpret_cast<const ulonglong2 *>(cut.boxes);
    if (wait) pdl_wait();
    pdl_trigger();
    // staging: entry e of table T (numbered over all levels) goes to 16-byte units 3 * e + T + 1 .. + 3 in the oriented form;
    // unit 3 * (first entry of T) + T holds the table's entry count.  The extra unit per table also spreads the tables over
    // the banks (without it the tables of a level are a power-of-two number of bytes apart and lanes that read different
    // tables would all hit the same banks).
    float4 *s_unit = reinterpret_cast<float4 *>(s_box);
    for (uint32_t e = threadIdx.x; e < smem_entries; e += blockDim.x) {
        uint32_t l = 0;
        while (l + 1 < cut.m && e >= cut.ent_off[l + 1]) ++l;
        const uint32_t in_level = e - cut.ent_off[l], T = cut.tab_off[l] + in_level / cut.w[l];
        const float4 A = cut.boxes[2 * (size_t)e], B = cut.boxes[2 * (size_t)e + 1];     // lo.x lo.y hi.x hi.y | lo.z hi.z cnt -
        float4 *u = s_unit + 3 * (size_t)e + T;
        if (in_level % cut.w[l] == 0) u[0] = make_float4(B.z, 0.f, 0.f, 0.f);      // the count (a bit pattern)
        u[1] = make_float4(A.x, A.z, -A.z, -A.x);
        u[2] = make_float4(A.y, A.w, -A.w, -A.y);
        u[3] = make_float4(B.x, B.y, -B.y, -B.x);
    }
    const uint32_t sa_box = (uint32_t)__cvta_generic_to_shared(s_box);
    __syncthreads();
    const uint64_t stride = (uint64_t)gridDim.x * blockDim.x;
    for (uint64_t ri = (uint64_t)blockIdx.x * blockDim.x + threadIdx.x; ri < n; ri += stride) {
        float4 a, b;
        ld_ray(rays + 2 * ri, a, b);
        RayEnc r;
        const float ix = 1.0f / b.x, iy = 1.0f / b.y, iz = 1.0f / b.z;
        r.oxy = pack2(a.x, a.y); r.ozz = pack2(a.z, a.z); r.tmin = a.w;
        r.ixy = pack2(ix, iy); r.izz = pack2(iz, iz); r.tmax = b.w;
        // the oriented form for the staged tables; a zero or NaN direction component (|inv| not finite) takes the generic test
        const bool plain = fabsf(ix) < __int_as_float(0x7f800000) && fabsf(iy) < __int_as_float(0x7f800000) &&
                           fabsf(iz) < __int_as_float(0x7f800000);
        RayOri q;
        {
            const bool nx = ix < 0.0f, ny = iy < 0.0f, nz = iz < 0.0f;
            const float ox = nx ? -a.x : a.x, oy = ny ? -a.y : a.y, oz = nz ? -a.z : a.z;
            q.ox = pack2(ox, ox); q.oy = pack2(oy, oy); q.oz = pack2(oz, oz);
            q.ix = pack2(fabsf(ix), fabsf(ix)); q.iy = pack2(fabsf(iy), fabsf(iy)); q.iz = pack2(fabsf(iz), fabsf(iz));
            q.bx = nx ? 8u : 0u; q.by = ny ? 24u : 16u; q.bz = nz ? 40u : 32u;
        }
        unsigned long long key = 0;
        uint32_t table = 0;
        bool alive = true;
        for (uint32_t l = 0; l < cut.m; ++l) {
            const uint32_t w = cut.w[l];
            unsigned long long mask = 0;
            if (alive) {
                const uint32_t e0 = cut.ent_off[l] + table * w;
                const bool in_smem = e0 < smem_entries;           // uniform per level
                const ulonglong2 *box = g_box + 2 * (size_t)e0;
                const uint32_t cnt_at = sa_box + 16u * (3u * e0 + cut.tab_off[l] + table), ent = cnt_at + 16u;
                uint32_t cnt;
                if (in_smem) asm volatile("ld.shared.u32 %0, [%1];" : "=r"(cnt) : "r"(cnt_at));
                else cnt = (uint32_t)ldg_u2(box + 1).y;           // low word = count
                // entries [0,cnt) are valid; entry j -> bit (w-1-j)
                uint32_t c_hi = cnt > 32u ? cnt - 32u : 0u;       // only flat tables wider than 32
                unsigned long long m_hi = 0;
                uint32_t m_lo;
                if (in_smem) {
                    if (plain) {
                        if (c_hi) m_hi = staged_mask(q, r.tmin, r.tmax, ent, 0, c_hi);
                        m_lo = staged_mask(q, r.tmin, r.tmax, ent, c_hi, cnt);
                    } else {
                        if (c_hi) m_hi = staged_mask_generic(r, ent, 0, c_hi);
                        m_lo = staged_mask_generic(r, ent, c_hi, cnt);
                    }
                } else {
                    if (c_hi) m_hi = table_mask<false>(r, box, 0, c_hi);
                    m_lo = table_mask<false>(r, box, c_hi, cnt);
                }
                mask = (c_hi ? (m_hi << 32) : 0ull) | (unsigned long long)m_lo;   // cnt bits, entry 0 on top
                uint32_t rep = (uint32_t)__clzll((long long)mask) - (64u - cnt);  // first hit entry (mask != 0)
                mask = cnt ? mask << (w - cnt) : 0ull;            // cnt >= 1 keeps the shift below 64
                if (mask == 0ull) alive = false; else table = table * w + rep;
            }
            key = (w < 64u ? key << w : 0ull) | mask;
        }
        keys[ri] = (KeyT)key;
    }
}

// TwoPoint: quantise o and o + len*d to b bits per coordinate, interleave.
__device__ __forceinline__ uint32_t quantise(float p, float lo, float hi, float scale, uint32_t qmax) {
    float ext = hi - lo;
    if (!(ext > 0.0f)) return 0u;
    float x = ((p - lo) / ext) * scale;
    if (!(x >= 0.0f)) return 0u;
    if (x >= scale) return qmax;
    return (uint32_t)x;
}

// spread5[x]: bit i of the 5-bit x at bit 6 * i (the Morton stride of six interleaved coordinates)
__device__ __forceinline__ uint32_t spread5_of(uint32_t x) {
    return (x & 1u) | ((x & 2u) << 5) | ((x & 4u) << 10) | ((x & 8u) << 15) | ((x & 16u) << 20);
}

template <typename KeyT>
__global__ void __launch_bounds__(ENC_THREADS)
k_encode_twopoint(const float4 *__restrict__ rays, uint64_t n, float3 lo, float3 hi, float len, uint32_t b,
                  KeyT *__restrict__ keys, int wait) {
    // the interleave as table look-ups: 32 words, one per bank, so any mix of indices in a warp is conflict-free
    __shared__ uint32_t s_spread[32];
    if (threadIdx.x < 32) s_spread[threadIdx.x] = spread5_of(threadIdx.x);
    if (wait) pdl_wait();
    pdl_trigger();
    __syncthreads();
    const uint64_t stride = (uint64_t)gridDim.x * ENC_THREADS;
    const float scale = (float)(1u << b);
    const uint32_t qmax = (1u << b) - 1u;
    uint64_t ri = (uint64_t)blockIdx.x * ENC_THREADS + threadIdx.x;
    float4 no = make_float4(0.f, 0.f, 0.f, 0.f), nd = no;
    if (ri < n) ld_ray(rays + 2 * ri, no, nd);
    for (; ri < n; ri += stride) {
        const float4 o = no, d = nd;
        if (ri + stride < n) ld_ray(rays + 2 * (ri + stride), no, nd);     // the next ray arrives while this one is coded
        uint32_t q[6];
        q[0] = quantise(o.x, lo.x, hi.x, scale, qmax);
        q[1] = quantise(o.y, lo.y, hi.y, scale, qmax);
        q[2] = quantise(o.z, lo.z, hi.z, scale, qmax);
        q[3] = quantise(o.x + len * d.x, lo.x, hi.x, scale, qmax);
        q[4] = quantise(o.y + len * d.y, lo.y, hi.y, scale, qmax);
        q[5] = quantise(o.z + len * d.z, lo.z, hi.z, scale, qmax);
        // coordinate c's bit i sits at key bit 6 * i + (5 - c): o.x first from the top (R10); b <= 10
        unsigned long long key = 0;
#pragma unroll
        for (int c = 0; c < 6; ++c) {
            unsigned long long s_ = s_spread[q[c] & 31u];
            if (sizeof(KeyT) == 8) s_ |= (unsigned long long)s_spread[(q[c] >> 5) & 31u] << 30;
            key |= s_ << (5 - c);
        }
        keys[ri] = (KeyT)key;
    }
}

// (f3) prefix path code, PAPER.md:116-128 (Figure 5); the walk is stated in include/hcc.h.
// One ray per thread, depth-first with the left child first over the canonical fp32 nodes; each
// popped node's slab test (the same arithmetic as slab_hit above) appends one bit.
constexpr int PPC_STACK = 66;   // depth <= 63 (hcc_bvh_create): at most depth + 1 pending nodes
template <typename KeyT>
__global__ void __launch_bounds__(ENC_THREADS)
k_encode_ppc(const float4 *__restrict__ rays, uint64_t n, const float4 *__restrict__ nodes, uint32_t bits,
             KeyT *__restrict__ keys) {
    pdl_wait();
    pdl_trigger();
    const uint64_t stride = (uint64_t)gridDim.x * blockDim.x;
    for (uint64_t ri = (uint64_t)blockIdx.x * blockDim.x + threadIdx.x; ri < n; ri += stride) {
        float4 a, b;
        ld_ray(rays + 2 * ri, a, b);
        RayEnc r;
        const float iz = 1.0f / b.z;
        r.oxy = pack2(a.x, a.y); r.ozz = pack2(a.z, a.z); r.tmin = a.w;
        r.ixy = pack2(1.0f / b.x, 1.0f / b.y); r.izz = pack2(iz, iz); r.tmax = b.w;
        uint32_t stack[PPC_STACK];
        int sp = 0;
        unsigned long long key = 0;
        uint32_t done = 0;
        stack[sp++] = 0u;
        while (sp > 0 && done < bits) {
            const uint32_t i = stack[--sp];
            const float4 n0 = __ldg(nodes + 2 * (size_t)i), n1 = __ldg(nodes + 2 * (size_t)i + 1);   // lo.xyz hi.x | hi.yz left count
            ulonglong2 A;
            A.x = pack2(n0.x, n0.y); A.y = pack2(n0.w, n1.x);
            const bool hit = slab_hit(r, A, pack2(n0.z, n1.y));
            key = (key << 1) | (hit ? 1ull : 0ull);
            ++done;
            if (hit && __float_as_uint(n1.w) == 0u) {
                const uint32_t left = __float_as_uint(n1.z);
                stack[sp++] = left + 1u;
                stack[sp++] = left;
            }
        }
        keys[ri] = (KeyT)(done < bits ? key << (bits - done) : key);
    }
}

// CTAs per SM of `kernel` at (threads, smem), queried once per device and configuration
static int ctas_per_sm(const void *kernel, int threads, size_t smem) {
    struct Entry { const void *k; int dev, threads; size_t smem; int per_sm; };
    static Entry cache[32];
    static std::atomic<int> used{0};
    const int dev = current_device();
    const int n = used.load(std::memory_order_acquire);
    for (int i = 0; i < n; ++i)
        if (cache[i].k == kernel && cache[i].dev == dev && cache[i].threads == threads && cache[i].smem == smem) return cache[i].per_sm;
    int per_sm = 1;
    if (cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, kernel, threads, smem) != cudaSuccess || per_sm < 1) per_sm = 1;
    static std::atomic_flag busy = ATOMIC_FLAG_INIT;
    if (!busy.test_and_set(std::memory_order_acquire)) {       // best effort: a lost race only repeats the query
        const int m = used.load(std::memory_order_relaxed);
        if (m < 32) { cache[m] = Entry{kernel, dev, threads, smem, per_sm}; used.store(m + 1, std::memory_order_release); }
        busy.clear(std::memory_order_release);
    }
    return per_sm;
}

static int grid_for(const void *kernel, size_t smem, uint64_t n, int threads = ENC_THREADS) {
    const int per_sm = ctas_per_sm(kernel, threads, smem);
    uint64_t want = (n + threads - 1) / threads;
    uint64_t cap = (uint64_t)sm_count() * (uint64_t)per_sm;
    return (int)(want < cap ? want : cap);
}

// the dynamic shared-memory limit of the HCC encoder, raised once per device
template <typename KeyT>
static cudaError_t encode_attr(size_t budget) {
    static std::atomic<int> done[HCC_MAX_DEVICES];
    const int dev = current_device();
    if (done[dev].load(std::memory_order_acquire)) return cudaSuccess;
    cudaError_t e = cudaFuncSetAttribute(k_encode_hcc<KeyT>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)budget);
    if (e == cudaSuccess) done[dev].store(1, std::memory_order_release);
    return e;
}

}  // namespace hcc

using namespace hcc;

int32_t hcc::encode_launch(const float *rays_dev, uint64_t n, const hcc_cut *cut, void *keys_dev, cudaStream_t s, LaunchKind kind) {
    HCC_REQUIRE(cut && cut->valid, HCC_ERR_INVALID_ARG, "hcc_encode: the cut handle holds no selection");
    if (n == 0) return HCC_OK;
    HCC_REQUIRE(rays_dev && keys_dev, HCC_ERR_INVALID_ARG, "hcc_encode: NULL argument");
    HCC_REQUIRE(aligned(rays_dev, 32) && aligned(keys_dev, 16), HCC_ERR_BAD_ALIGNMENT,
                "hcc_encode: rays need 32-byte, keys 16-byte alignment");
    HCC_REQUIRE(n < (1ull << 32), HCC_ERR_UNSUPPORTED, "hcc_encode: n >= 2^32");
    const CutDev &d = cut->dev;
    // stage whole levels, top down, while they fit in 160 KB (leaves room for 1 CTA/SM at worst)
    const size_t budget = HCC_ENC_STAGE_BYTES;
    uint32_t smem_entries = 0;
    uint32_t smem_tables = 0;
    for (uint32_t l = 0; l < d.m; ++l) {
        uint32_t end = d.ent_off[l] + d.n_tab[l] * d.w[l];
        if ((size_t)end * 48 + (size_t)(d.tab_off[l] + d.n_tab[l]) * 16 <= budget) { smem_entries = end; smem_tables = d.tab_off[l] + d.n_tab[l]; }
        else break;
    }
    size_t smem = (size_t)smem_entries * 48 + (size_t)smem_tables * 16;     // oriented entries of 48 bytes + one unit per staged table
    if (cut->container_bits == 32) {
        auto kern = k_encode_hcc<uint32_t>;
        HCC_CUDA_TRY(encode_attr<uint32_t>(budget));
        HCC_CUDA_TRY(launch_k(kind, kern, dim3(grid_for((const void *)kern, smem, n, ENC_HCC_THREADS)), dim3(ENC_HCC_THREADS), smem, s,
                              (const float4 *)rays_dev, n, d, smem_entries, (uint32_t *)keys_dev, kind_waits(kind)));
    } else {
        auto kern = k_encode_hcc<unsigned long long>;
        HCC_CUDA_TRY(encode_attr<unsigned long long>(budget));
        HCC_CUDA_TRY(launch_k(kind, kern, dim3(grid_for((const void *)kern, smem, n, ENC_HCC_THREADS)), dim3(ENC_HCC_THREADS), smem, s,
                              (const float4 *)rays_dev, n, d, smem_entries, (unsigned long long *)keys_dev, kind_waits(kind)));
    }
    return HCC_OK;
}

extern "C" int32_t hcc_encode(const float *rays_dev, uint64_t n, const hcc_cut *cut, void *keys_dev, void *stream) {
    return encode_launch(rays_dev, n, cut, keys_dev, (cudaStream_t)stream, LK_FIRST);
}

int32_t hcc::encode_twopoint_launch(const float *rays_dev, uint64_t n, const float scene_lo[3], const float scene_hi[3],
                                    uint32_t key_bits, void *keys_dev, cudaStream_t s, LaunchKind kind) {
    HCC_REQUIRE(key_bits == 16 || key_bits == 24 || key_bits == 32 || key_bits == 48 || key_bits == 64,
                HCC_ERR_INVALID_ARG, "hcc_encode_twopoint: key_bits must be 16, 24, 32, 48 or 64");
    if (n == 0) return HCC_OK;
    HCC_REQUIRE(rays_dev && keys_dev && scene_lo && scene_hi, HCC_ERR_INVALID_ARG, "hcc_encode_twopoint: NULL argument");
    HCC_REQUIRE(aligned(rays_dev, 32) && aligned(keys_dev, 16), HCC_ERR_BAD_ALIGNMENT,
                "hcc_encode_twopoint: rays need 32-byte, keys 16-byte alignment");
    float3 lo = make_float3(scene_lo[0], scene_lo[1], scene_lo[2]);
    float3 hi = make_float3(scene_hi[0], scene_hi[1], scene_hi[2]);
    float e = fmaxf(fmaxf(hi.x - lo.x, hi.y - lo.y), hi.z - lo.z);
    float len = 0.25f * e;
    uint32_t b = key_bits / 6u;
    if (key_bits <= 32) {
        auto kern = k_encode_twopoint<uint32_t>;
        HCC_CUDA_TRY(launch_k(kind, kern, dim3(grid_for((const void *)kern, 0, n)), dim3(ENC_THREADS), 0, s,
                                (const float4 *)rays_dev, n, lo, hi, len, b, (uint32_t *)keys_dev, kind_waits(kind)));
    } else {
        auto kern = k_encode_twopoint<unsigned long long>;
        HCC_CUDA_TRY(launch_k(kind, kern, dim3(grid_for((const void *)kern, 0, n)), dim3(ENC_THREADS), 0, s,
                                (const float4 *)rays_dev, n, lo, hi, len, b, (unsigned long long *)keys_dev, kind_waits(kind)));
    }
    return HCC_OK;
}

extern "C" int32_t hcc_encode_twopoint(const float *rays_dev, uint64_t n, const float scene_lo[3], const float scene_hi[3],
                                       uint32_t key_bits, void *keys_dev, void *stream) {
    return encode_twopoint_launch(rays_dev, n, scene_lo, scene_hi, key_bits, keys_dev, (cudaStream_t)stream, LK_FIRST);
}

extern "C" int32_t hcc_encode_ppc(const hcc_bvh *bvh, const float *rays_dev, uint64_t n, uint32_t key_bits, void *keys_dev,
                                  void *stream) {
    HCC_REQUIRE(bvh, HCC_ERR_INVALID_ARG, "hcc_encode_ppc: NULL bvh");
    HCC_REQUIRE(key_bits == 16 || key_bits == 24 || key_bits == 32 || key_bits == 48 || key_bits == 64,
                HCC_ERR_INVALID_ARG, "hcc_encode_ppc: key_bits must be 16, 24, 32, 48 or 64");
    if (n == 0) return HCC_OK;
    HCC_REQUIRE(rays_dev && keys_dev, HCC_ERR_INVALID_ARG, "hcc_encode_ppc: NULL argument");
    HCC_REQUIRE(aligned(rays_dev, 32) && aligned(keys_dev, 16), HCC_ERR_BAD_ALIGNMENT,
                "hcc_encode_ppc: rays need 32-byte, keys 16-byte alignment");
    HCC_REQUIRE(n < (1ull << 32), HCC_ERR_UNSUPPORTED, "hcc_encode_ppc: n >= 2^32");
    cudaStream_t s = (cudaStream_t)stream;
    const float4 *nodes = reinterpret_cast<const float4 *>(bvh->d_nodes);
    if (key_bits <= 32) {
        auto kern = k_encode_ppc<uint32_t>;
        HCC_CUDA_TRY(launch_k(LK_FIRST, kern, dim3(grid_for((const void *)kern, 0, n)), dim3(ENC_THREADS), 0, s, (const float4 *)rays_dev, n, nodes, key_bits, (uint32_t *)keys_dev));
    } else {
        auto kern = k_encode_ppc<unsigned long long>;
        HCC_CUDA_TRY(launch_k(LK_FIRST, kern, dim3(grid_for((const void *)kern, 0, n)), dim3(ENC_THREADS), 0, s, (const float4 *)rays_dev, n, nodes, key_bits, (unsigned long long *)keys_dev));
    }
    HCC_CUDA_TRY(cudaGetLastError());
    return HCC_OK;
}
