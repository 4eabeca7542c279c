// (a4) trace: software BVH traversal of the (re)ordered rays — PAPER.md:247 ("the trace
// kernel fetches the rays based on these sorted indices"), :62-64.  B200 has no RT cores.
//
// Design: persistent warps pull 32-ray chunks of the (sorted) order from an
// atomic counter and refill finished lanes from the same chunk, so the rays of a warp stay
// neighbours in the sorted order.  A warp alternates between
//  - node steps: every lane that holds a reference to a wide node fetches its 64-byte record
//    (bvh.cu: four quantised child boxes + four references, two 256-bit loads) and tests the four
//    boxes.  Hit LEAF children are not visited by the lane: it appends (leaf, owner lane) entries to
//    the warp's leaf queue in shared memory (slots handed out by one shared-memory atomic add), so
//    neither the traversal stack nor `cur` ever holds a leaf and a lane never waits for a triangle
//    test.  Hit INTERNAL children are ordered by entry distance: the nearest is next, the others
//    are pushed.  Node steps repeat with two warp votes per step until a round of leaves waits;
//  - triangle rounds: the WHOLE warp tests the leaves at the head of the queue, TRI_LPL lanes per
//    leaf, whoever owns the rays: the ray of a leaf is read from its owner's shared-memory slot, a
//    hit is committed there with a 64-bit atomic min on (t, prim) (closest hit) or a flag store
//    (any hit); the owners refresh their culling distance afterwards;
//  - retire + refill, batched: only when REFILL_AT lanes are finished (or nothing else can run)
//    are their hits written and new rays loaded.
// A ray is finished when its stack is empty and its queued leaves have been tested.  The traversal
// stack lives in shared memory (conflict-free) and spills to local memory.
// Compiled with -fmad=false; fmaf() appears exactly where hcc.h states it for the triangle
// predicate, which alone defines the results.
#include "common.cuh"

namespace hcc {

#ifndef HCC_TRACE_THREADS             // threads of a CTA: 32, 64 or 128 (the warps of a CTA share nothing but its lifetime)
#define HCC_TRACE_THREADS 128
#endif
constexpr int TRACE_THREADS = HCC_TRACE_THREADS;
#ifndef HCC_TRACE_BLOCKS_PER_SM       // closest hit: CTAs per SM
#define HCC_TRACE_BLOCKS_PER_SM (7 * 128 / HCC_TRACE_THREADS)
#endif
#ifndef HCC_TRACE_BLOCKS_PER_SM_ANY
#define HCC_TRACE_BLOCKS_PER_SM_ANY (7 * 128 / HCC_TRACE_THREADS)
#endif
#ifndef HCC_TRACE_REFILL_AT
#define HCC_TRACE_REFILL_AT 8
#endif
#ifndef HCC_TRACE_SMEM_STACK
#define HCC_TRACE_SMEM_STACK 16
#endif
#ifndef HCC_TRACE_WALK_MIN            // with fewer lanes able to take a node step the leaf queue is drained first
#define HCC_TRACE_WALK_MIN 8
#endif
#ifndef HCC_TRACE_ANY_ORDERED         // any hit: 1 = nearest child first (as closest hit), 0 = first hit child in slot order
#define HCC_TRACE_ANY_ORDERED 1
#endif
#ifndef HCC_TRACE_LPL                 // lanes per leaf in a triangle round (4, 2 or 1): a round tests 32 / LPL leaves
#define HCC_TRACE_LPL 2
#endif
#ifndef HCC_TRACE_LPL_ANY
#define HCC_TRACE_LPL_ANY 2
#endif
constexpr int TRACE_BLOCKS_PER_SM = HCC_TRACE_BLOCKS_PER_SM, TRACE_BLOCKS_PER_SM_ANY = HCC_TRACE_BLOCKS_PER_SM_ANY;
constexpr int SMEM_STACK = HCC_TRACE_SMEM_STACK;   // entries per thread in shared memory
constexpr int STACK_SIZE = 3 * 64 + 4;  // hcc_bvh_create admits depth <= 63 (+1 for a split leaf); a 4-wide step pushes at most 3
constexpr uint32_t CHUNK = 32;          // rays a warp takes from the counter at a time
constexpr uint32_t REFILL_AT = HCC_TRACE_REFILL_AT;   // finished lanes that trigger retirement + refill
constexpr int TRACE_WARPS = TRACE_THREADS / 32;
// leaf queue entries per warp, a power of two: a node step appends at most 4 x 32 entries and starts with
// fewer than a round's worth (<= 32) waiting
constexpr uint32_t QCAP = 256;

// Shared memory of a CTA, addressed with 32-bit shared-window addresses:
//   lane slots : 48 bytes per thread: ray (o, tmin | d, t_best) at +0 / +16 (t_best starts as tmax and is
//                lowered by committed hits), closest: key ord(t) << 32 | prim at +32 and (u, v) at +40;
//                any: occluded flag at +32
//   leaf queues: QCAP x 8 bytes per warp: (leaf reference, owner lane); queue tails: one word per warp
//   stacks     : SMEM_STACK rows of one word per thread (a lane's entries are ROW bytes apart: conflict-free)
constexpr uint32_t SLOT_BYTES = 48;
constexpr uint32_t ROW = 4u * TRACE_THREADS, ROW_SHIFT = TRACE_THREADS == 128 ? 9u : TRACE_THREADS == 64 ? 8u : 7u;
static_assert(TRACE_THREADS == 32 || TRACE_THREADS == 64 || TRACE_THREADS == 128, "CTA size");
constexpr uint32_t OFF_SLOTS = 0, OFF_QUEUE = OFF_SLOTS + SLOT_BYTES * TRACE_THREADS,
                   OFF_TAIL = OFF_QUEUE + 8 * QCAP * TRACE_WARPS, OFF_STACK = OFF_TAIL + 16,
                   SMEM_BYTES = OFF_STACK + ROW * SMEM_STACK;
static_assert(TRACE_WARPS <= 4, "queue tails: one word per warp in 16 bytes");

__device__ __forceinline__ uint32_t lds32(uint32_t a) { uint32_t v; asm volatile("ld.shared.u32 %0, [%1];" : "=r"(v) : "r"(a) : "memory"); return v; }
__device__ __forceinline__ void sts32(uint32_t a, uint32_t v) { asm volatile("st.shared.u32 [%0], %1;" ::"r"(a), "r"(v) : "memory"); }
__device__ __forceinline__ uint2 lds64(uint32_t a) { uint2 v; asm volatile("ld.shared.v2.u32 {%0,%1}, [%2];" : "=r"(v.x), "=r"(v.y) : "r"(a) : "memory"); return v; }
__device__ __forceinline__ void sts64(uint32_t a, uint32_t x, uint32_t y) { asm volatile("st.shared.v2.u32 [%0], {%1,%2};" ::"r"(a), "r"(x), "r"(y) : "memory"); }
__device__ __forceinline__ float4 lds128(uint32_t a) {
    float4 v;
    asm volatile("ld.shared.v4.f32 {%0,%1,%2,%3}, [%4];" : "=f"(v.x), "=f"(v.y), "=f"(v.z), "=f"(v.w) : "r"(a) : "memory");
    return v;
}
__device__ __forceinline__ void sts128(uint32_t a, float4 v) {
    asm volatile("st.shared.v4.f32 [%0], {%1,%2,%3,%4};" ::"r"(a), "f"(v.x), "f"(v.y), "f"(v.z), "f"(v.w) : "memory");
}
__device__ __forceinline__ void atom_min64(uint32_t a, unsigned long long v) {
    asm volatile("red.shared.min.u64 [%0], %1;" ::"r"(a), "l"(v) : "memory");
}

__device__ __forceinline__ uint32_t atom_add32(uint32_t a, uint32_t v) {
    uint32_t old;
    asm volatile("atom.shared.add.u32 %0, [%1], %2;" : "=r"(old) : "r"(a), "r"(v) : "memory");
    return old;
}

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

// float bits <-> unsigned keys of the same order (negative t included)
__device__ __forceinline__ uint32_t ord_of(float f) {
    const uint32_t b = __float_as_uint(f);
    return b ^ ((uint32_t)((int32_t)b >> 31) | 0x80000000u);
}
__device__ __forceinline__ float float_of(uint32_t k) {
    return __uint_as_float(k ^ (((k >> 31) - 1u) | 0x80000000u));
}

// The triangle predicate of hcc.h, operation by operation, with the upper end left to the caller:
// true <=> det != 0, u >= 0, v >= 0, u + v <= 1, t > tmin.   o = (ox, oy, oz, tmin), d = (dx, dy, dz, -).
__device__ __forceinline__ bool tri_hit(const float4 o, const float4 d, const float4 v0, const float4 e1, const float4 e2,
                                        float &t, float &u, float &v) {
    float px = fmaf(d.y, e2.z, -(d.z * e2.y));
    float py = fmaf(d.z, e2.x, -(d.x * e2.z));
    float pz = fmaf(d.x, e2.y, -(d.y * e2.x));
    float det = fmaf(e1.x, px, fmaf(e1.y, py, e1.z * pz));
    if (det == 0.0f) return false;
    float inv = 1.0f / det;
    float sx = o.x - v0.x, sy = o.y - v0.y, sz = o.z - v0.z;
    u = fmaf(sx, px, fmaf(sy, py, sz * pz)) * inv;
    if (!(u >= 0.0f)) return false;
    float qx = fmaf(sy, e1.z, -(sz * e1.y));
    float qy = fmaf(sz, e1.x, -(sx * e1.z));
    float qz = fmaf(sx, e1.y, -(sy * e1.x));
    v = fmaf(d.x, qx, fmaf(d.y, qy, d.z * qz)) * inv;
    if (!(v >= 0.0f) || !(u + v <= 1.0f)) return false;
    t = fmaf(e2.x, qx, fmaf(e2.y, qy, e2.z * qz)) * inv;
    return t > o.w;
}

struct TraceScene {
    const uint32_t *wrec;
    const float4 *ttri;
    uint32_t root_ref;
    uint32_t wait;      // call griddepcontrol.wait before the first global access (0: a dependent launch that overlaps its predecessor)
    float q_lo[3], q_scale[3];
};

// ctl[0] = next ray rank (zeroed on the launch stream before every launch).
// STATS: the same traversal also counts the wide-node records fetched (64 bytes each) and the
// triangle records fetched (64 bytes each): stats[0], stats[1]; stats[2] = rays, stats[3] =
// deepest stack seen; stats[4] = distinct node records summed over warp-level node steps (what
// a coherent warp saves), stats[5] = warp-level node steps, stats[6] = lanes taking part in
// them, stats[7] = warp-level triangle rounds (stats[1] / stats[7] = triangle tests per round; a lane may test
// several triangles of its leaf in one round, so this can exceed 32).
// Used for the diagnostics only, never timed.
template <bool ANY, bool STATS>
__global__ void __launch_bounds__(TRACE_THREADS, ANY ? TRACE_BLOCKS_PER_SM_ANY : TRACE_BLOCKS_PER_SM)
k_trace(const TraceScene sc, const float4 *__restrict__ rays, const uint32_t *__restrict__ perm, uint32_t n,
        void *__restrict__ hits, uint32_t *ctl, unsigned long long *stats) {
    constexpr uint32_t LPL = ANY ? HCC_TRACE_LPL_ANY : HCC_TRACE_LPL;     // lanes per leaf in a triangle round
    constexpr uint32_t ROUND_LEAVES = 32u / LPL;
    static_assert(LPL == 1 || LPL == 2 || LPL == 4, "lanes per leaf");
    __shared__ __align__(16) unsigned char smem[SMEM_BYTES];
    uint32_t l_stack[STACK_SIZE - SMEM_STACK];
    const uint32_t tid = threadIdx.x, lane = tid & 31u;
    const uint32_t lanes_below = (1u << lane) - 1u;
    const uint32_t sa = (uint32_t)__cvta_generic_to_shared(smem);
    const uint32_t sa_slot = sa + OFF_SLOTS + SLOT_BYTES * tid;                  // this lane's slot
    const uint32_t sa_wslots = sa + OFF_SLOTS + SLOT_BYTES * (tid & ~31u);       // slot of lane 0 of the warp
    const uint32_t sa_queue = sa + OFF_QUEUE + 8u * QCAP * (tid >> 5);
    const uint32_t sa_tail = sa + OFF_TAIL + 4u * (tid >> 5);
    const uint32_t st_base = sa + OFF_STACK + 4u * tid, st_limit = st_base + ROW * SMEM_STACK;
    unsigned long long n_nodes = 0, n_tris = 0, n_rays = 0, n_sect = 0, n_steps = 0, n_lanes = 0, n_rounds = 0;
    uint32_t max_sp = 0;

    uint32_t w_next = 0, w_end = 0;      // the warp's current chunk of ranks
    uint32_t q_head = 0, q_tail = 0;     // leaf queue positions (warp-uniform, monotonic); the tail's master copy is in shared memory
    bool exhausted = false, have = false;
    uint32_t cur = 0, rid = 0;           // cur: 0 = nothing left to walk, else the reference of a wide node
    uint32_t pend_end = 0;               // queue position behind the lane's last queued leaf
    uint32_t sp = st_base;               // address of the next free stack entry (rows beyond st_limit live in l_stack)
    float tmin = 0.f;
    float ix = 0.f, iy = 0.f, iz = 0.f;                                 // slab planes: t = (32768 + cell) * i + c
    float cnx = 0.f, cny = 0.f, cnz = 0.f, cfx = 0.f, cfy = 0.f, cfz = 0.f;   // c of the near / far planes
    uint32_t snx = SEL_LO, sny = SEL_LO, snz = SEL_LO;                  // near-plane selectors
    float best_t = 0.f;                                                 // culling limit
    const float INF = __int_as_float(0x7f800000);

    if (lane == 0) sts32(sa_tail, 0u);
    __syncwarp();
    if (sc.wait) pdl_wait();   // the permutation (or whatever wrote the rays) and the zeroed work counter are complete
    pdl_trigger();
#ifdef HCC_TRACE_TIMELINE   // debug builds only: per-warp start / exhaustion / end times behind the eight counters
    unsigned long long tl_t0 = 0, tl_ex = 0;
    if (stats) asm volatile("mov.u64 %0, %%globaltimer;" : "=l"(tl_t0));
#endif

    auto push = [&](uint32_t v) {      // general form (the node step has its own fast path)
        if (sp < st_limit) sts32(sp, v); else l_stack[(sp - st_limit) >> ROW_SHIFT] = v;
        sp += ROW;
    };
    auto pop = [&]() -> uint32_t {
        if (sp == st_base) return 0u;
        sp -= ROW;
        return sp < st_limit ? lds32(sp) : l_stack[(sp - st_limit) >> ROW_SHIFT];
    };

    // one triangle round: the ROUND_LEAVES leaves at the head of the queue, LPL lanes per leaf; lane k of a
    // leaf tests its triangles k, k + LPL, ... and commits the best of them
    auto tri_round = [&]() {
        const uint32_t pos = q_head + lane / LPL;
        const bool valid = (int32_t)(q_tail - pos) > 0;
        const uint2 e = lds64(sa_queue + 8u * (pos & (QCAP - 1u)));      // (leaf reference, owner lane); stale if !valid
        const uint32_t last = (e.x >> 28) & 7u;                          // triangles of the leaf - 1
        const uint32_t sa_own = sa_wslots + SLOT_BYTES * e.y;
        bool hit = false;
        float t = 0.f, u = 0.f, v = 0.f;
        uint32_t prim = 0u;
        uint32_t k = lane % LPL;
        if (valid && k <= last) {
            const float4 ro = lds128(sa_own), rd = lds128(sa_own + 16u);
            const float4 *tp = sc.ttri + 4 * (size_t)((e.x & 0x0FFFFFFFu) + k);
#pragma unroll 1
            for (;;) {
                const Words8 T = ld256(reinterpret_cast<const uint32_t *>(tp));
                const float4 e2 = __ldg(tp + 2);
                const float4 v0 = make_float4(__uint_as_float(T.w[0]), __uint_as_float(T.w[1]), __uint_as_float(T.w[2]), 0.f);
                const float4 e1 = make_float4(__uint_as_float(T.w[4]), __uint_as_float(T.w[5]), __uint_as_float(T.w[6]), 0.f);
                float t1, u1, v1;
                // closest: rd.w is the best t so far (tmax at first): later hits lose anyway, equal ones go to the key
                if (tri_hit(ro, rd, v0, e1, e2, t1, u1, v1) && (ANY ? t1 < rd.w : t1 <= rd.w)) {
                    // the lane's own triangles: nearest first, equal t to the lower prim id
                    if (ANY || !hit || t1 < t || (t1 == t && T.w[3] < prim)) { t = t1; u = u1; v = v1; prim = T.w[3]; }
                    hit = true;
                }
                if (STATS) ++n_tris;
                if (LPL == 4) break;
                k += LPL;
                if (k > last || (ANY && hit)) break;
                tp += 4 * LPL;
            }
        }
        if (ANY) {
            if (hit) sts32(sa_own + 32u, 1u);
        } else if (__any_sync(0xFFFFFFFFu, hit)) {
            const unsigned long long key = ((unsigned long long)ord_of(t) << 32) | prim;
            if (hit) atom_min64(sa_own + 32u, key);
            __syncwarp();
            if (hit) {
                const uint2 now = lds64(sa_own + 32u);
                if (now.x == prim && now.y == (uint32_t)(key >> 32)) {   // this lane's hit is the best: publish t, u, v
                    sts32(sa_own + 28u, __float_as_uint(t));
                    sts64(sa_own + 40u, __float_as_uint(u), __float_as_uint(v));
                }
            }
        }
        if (STATS && lane == 0) ++n_rounds;
        q_head += min(ROUND_LEAVES, q_tail - q_head);
    };

    for (;;) {
        // ---- retire finished rays and refill their lanes, in batches of REFILL_AT (or when nothing else can run)
        {
            const bool done = have && cur == 0u && (int32_t)(q_head - pend_end) >= 0;
            const uint32_t free_m = __ballot_sync(0xFFFFFFFFu, done || !have);
            if (free_m == 0xFFFFFFFFu || (uint32_t)__popc(free_m) >= REFILL_AT) {
                if (done) {
                    if (ANY) reinterpret_cast<uint8_t *>(hits)[rid] = lds32(sa_slot + 32u) ? 1 : 0;
                    else {
                        const uint2 key = lds64(sa_slot + 32u);           // (prim, ord(t))
                        const bool hit = key.x != HCC_MISS_PRIM;
                        const uint2 uv = lds64(sa_slot + 40u);
                        reinterpret_cast<float4 *>(hits)[rid] =
                            make_float4(hit ? float_of(key.y) : INF, __uint_as_float(key.x), hit ? __uint_as_float(uv.x) : 0.f,
                                        hit ? __uint_as_float(uv.y) : 0.f);
                    }
                    have = false;
                }
                uint32_t idle = free_m;
                while (!exhausted && idle) {
                    if (w_next == w_end) {
                        uint32_t base = 0;
                        if (lane == 0) base = atomicAdd(&ctl[0], CHUNK);
                        base = __shfl_sync(0xFFFFFFFFu, base, 0);
                        if (base >= n) {
                            exhausted = true;
#ifdef HCC_TRACE_TIMELINE
                            if (stats) asm volatile("mov.u64 %0, %%globaltimer;" : "=l"(tl_ex));
#endif
                            break;
                        }
                        w_next = base;
                        w_end = min(base + CHUNK, n);
                    }
                    const uint32_t avail = w_end - w_next;
                    const uint32_t rank = __popc(idle & lanes_below);
                    if (!have && rank < avail) {
                        const uint32_t j = w_next + rank;
                        // a sorted order is walked from its END: hierarchy cut codes carry their densest cut nodes in
                        // the top bits, so the rays with the most traversal work start first and the kernel's tail
                        // (the last rays running alone) is made of cheap ones; a warp's rays stay neighbours
                        rid = perm ? ld_stream(perm + (n - 1u - j)) : j;
                        const float4 a = ld_stream4(rays + 2 * (size_t)rid), b = ld_stream4(rays + 2 * (size_t)rid + 1);
                        sts128(sa_slot, a);
                        sts128(sa_slot + 16u, b);
                        if (ANY) sts32(sa_slot + 32u, 0u);
                        else {
                            // every t < tmax gives a smaller key, every t >= tmax a larger one; low word = "no hit yet"
                            const unsigned long long k0 = ((unsigned long long)ord_of(b.w) << 32) - 1ull;
                            sts64(sa_slot + 32u, (uint32_t)k0, (uint32_t)(k0 >> 32));
                        }
                        tmin = a.w;
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
                        best_t = b.w;
                        sp = st_base;
                        cur = sc.root_ref;           // always a wide node (hcc_bvh_create)
                        pend_end = q_head;
                        have = true;
                        if (STATS) ++n_rays;
                    }
                    w_next += min((uint32_t)__popc(idle), avail);
                    idle = __ballot_sync(0xFFFFFFFFu, !have);
                }
                if (__ballot_sync(0xFFFFFFFFu, have) == 0u) break;
            }
        }

        // ---- node steps, until a round of leaves waits or too few lanes can walk
        uint32_t wm = __ballot_sync(0xFFFFFFFFu, cur != 0u);
        while (wm != 0u) {
            if (STATS) {
                const uint32_t peers = __match_any_sync(0xFFFFFFFFu, cur != 0u ? cur : (0x40000000u | lane));
                if (cur != 0u && (peers & lanes_below) == 0u) ++n_sect;
                if (lane == 0) { ++n_steps; n_lanes += __popc(wm); }
                max_sp = max(max_sp, (sp - st_base) >> ROW_SHIFT);
            }
            if (cur != 0u) {
                const uint32_t *rec = sc.wrec + 16 * (size_t)(cur - 1u);
                const Words8 A = ld256(rec), B = ld256(rec + 8);
                if (STATS) ++n_nodes;
                const uint32_t sfx = snx ^ SEL_FLIP, sfy = sny ^ SEL_FLIP, sfz = snz ^ SEL_FLIP;
                // child c: x, y, z words -> entry distance and "the ray meets the box before best_t"
#define HCC_BOX(X, Y, Z, D, H)                                                                                                           \
    {                                                                                                                                    \
        float tn = max3(fmaf(cell_plane(X, snx), ix, cnx), fmaf(cell_plane(Y, sny), iy, cny), fmaf(cell_plane(Z, snz), iz, cnz));         \
        float tf = min3(fmaf(cell_plane(X, sfx), ix, cfx), fmaf(cell_plane(Y, sfy), iy, cfy), fmaf(cell_plane(Z, sfz), iz, cfz));         \
        D = fmaxf(tn, tmin);                                                                                                             \
        tf = fminf(tf, best_t); /* a box starting AT best_t is kept */                                                                   \
        H = D <= tf;                                                                                                                     \
    }
                float d0, d1, d2, d3;
                bool h0, h1, h2, h3;
                HCC_BOX(A.w[0], A.w[1], A.w[2], d0, h0)
                HCC_BOX(A.w[3], A.w[4], A.w[5], d1, h1)
                HCC_BOX(A.w[6], A.w[7], B.w[0], d2, h2)
                HCC_BOX(B.w[1], B.w[2], B.w[3], d3, h3)
#undef HCC_BOX
                const uint32_t r0 = B.w[4], r1 = B.w[5], r2 = B.w[6], r3 = B.w[7];
                // hit leaves go to the warp's queue (slots from one shared-memory atomic add), never to the stack
                const bool l0 = h0 && (int32_t)r0 < 0, l1 = h1 && (int32_t)r1 < 0, l2 = h2 && (int32_t)r2 < 0, l3 = h3 && (int32_t)r3 < 0;
                const uint32_t nl = (l0 ? 1u : 0u) + (l1 ? 1u : 0u) + (l2 ? 1u : 0u) + (l3 ? 1u : 0u);
                if (nl != 0u) {
                    uint32_t pos = atom_add32(sa_tail, nl);
                    if (l0) { sts64(sa_queue + 8u * (pos & (QCAP - 1u)), r0, lane); ++pos; }
                    if (l1) { sts64(sa_queue + 8u * (pos & (QCAP - 1u)), r1, lane); ++pos; }
                    if (l2) { sts64(sa_queue + 8u * (pos & (QCAP - 1u)), r2, lane); ++pos; }
                    if (l3) { sts64(sa_queue + 8u * (pos & (QCAP - 1u)), r3, lane); ++pos; }
                    pend_end = pos;
                }
                // hit wide nodes: a missed child, a leaf and an unused slot (reference 0, never hit) get +inf
                d0 = h0 && (int32_t)r0 > 0 ? d0 : INF;
                d1 = h1 && (int32_t)r1 > 0 ? d1 : INF;
                d2 = h2 && (int32_t)r2 > 0 ? d2 : INF;
                d3 = h3 && (int32_t)r3 > 0 ? d3 : INF;
                uint32_t rW, rP0, rP1, rP2;          // next reference; pushed first .. last
                bool hW, hP0, hP1, hP2;
                if (!ANY || HCC_TRACE_ANY_ORDERED) {
                    // tournament: (0,1) -> A, loser L1; (2,3) -> B, loser L2; (A,B) -> nearest, loser L3.
                    // Pushed farthest-first by this partial order: the loser of the losing pair, the loser of
                    // the winning pair, then L3.
                    const bool s01 = d1 < d0, s23 = d3 < d2;
                    const float dA = s01 ? d1 : d0, dL1 = s01 ? d0 : d1;
                    const uint32_t rA = s01 ? r1 : r0, rL1 = s01 ? r0 : r1;
                    const float dB = s23 ? d3 : d2, dL2 = s23 ? d2 : d3;
                    const uint32_t rB = s23 ? r3 : r2, rL2 = s23 ? r2 : r3;
                    const bool sAB = dB < dA;
                    hW = (sAB ? dB : dA) < INF; rW = sAB ? rB : rA;
                    hP2 = (sAB ? dA : dB) < INF; rP2 = sAB ? rA : rB;
                    hP0 = (sAB ? dL1 : dL2) < INF; rP0 = sAB ? rL1 : rL2;     // pair losers: losing side first
                    hP1 = (sAB ? dL2 : dL1) < INF; rP1 = sAB ? rL2 : rL1;
                } else {
                    // slot order: the first hit child is next, the others are pushed
                    const bool i0 = d0 < INF, i1 = d1 < INF, i2 = d2 < INF, i3 = d3 < INF;
                    hW = i0 || i1 || i2 || i3;
                    rW = i0 ? r0 : i1 ? r1 : i2 ? r2 : r3;
                    hP2 = i0 && i1; rP2 = r1;
                    hP1 = (i0 || i1) && i2; rP1 = r2;
                    hP0 = (i0 || i1 || i2) && i3; rP0 = r3;
                }
                if (sp + 3u * ROW <= st_limit) {
                    // all in shared memory: store unconditionally, advance if the child was hit
                    sts32(sp, rP0); sp += hP0 ? ROW : 0u;
                    sts32(sp, rP1); sp += hP1 ? ROW : 0u;
                    sts32(sp, rP2); sp += hP2 ? ROW : 0u;
                    if (hW) cur = rW;
                    else if (sp == st_base) cur = 0u;
                    else { sp -= ROW; cur = lds32(sp); }
                } else {
                    if (hP0) push(rP0);
                    if (hP1) push(rP1);
                    if (hP2) push(rP2);
                    cur = hW ? rW : pop();
                }
            }
            __syncwarp();
            q_tail = lds32(sa_tail);
            wm = __ballot_sync(0xFFFFFFFFu, cur != 0u);
            if (q_tail - q_head >= ROUND_LEAVES || (uint32_t)__popc(wm) < HCC_TRACE_WALK_MIN) break;
        }

        // ---- triangle rounds: whenever a round's worth of leaves waits, or all of them when too few lanes can walk
        if (q_tail != q_head) {
            const bool drain = (uint32_t)__popc(wm) < HCC_TRACE_WALK_MIN;
            if (drain || q_tail - q_head >= ROUND_LEAVES) {
                do tri_round(); while (q_tail - q_head >= ROUND_LEAVES || (drain && q_tail != q_head));
                __syncwarp();
                if (have) {
                    if (ANY) { if (lds32(sa_slot + 32u)) { sp = st_base; cur = 0u; } }
                    else best_t = __uint_as_float(lds32(sa_slot + 28u));
                }
            }
        }
    }
    // A dependent launch that skipped the wait at entry (hcc_reorder_trace_pair's second traversal kernel) waits HERE, once
    // its own work is done: a dependent grid has to execute griddepcontrol.wait, and with it this grid cannot complete - and
    // nothing enqueued behind it on the stream can start - before the first batch's traversal kernel has completed and its
    // hits are visible.  The CTA only idles until then; every CTA of the primary grid is resident from the start (the grid
    // is capped at the resident CTAs), so a waiting CTA never stands in the way of one the primary still needs.
    if (!sc.wait) pdl_wait();
#ifdef HCC_TRACE_TIMELINE
    if (stats && lane == 0) {
        unsigned long long tl_t1;
        asm volatile("mov.u64 %0, %%globaltimer;" : "=l"(tl_t1));
        const size_t w = (size_t)blockIdx.x * TRACE_WARPS + (tid >> 5);
        stats[8 + 3 * w] = tl_t0; stats[9 + 3 * w] = tl_ex; stats[10 + 3 * w] = tl_t1;
    }
#endif
    if (STATS) {
        atomicAdd(&stats[0], n_nodes);
        atomicAdd(&stats[1], n_tris);
        atomicAdd(&stats[2], n_rays);
        atomicMax(&stats[3], (unsigned long long)max_sp);
        atomicAdd(&stats[4], n_sect);
        atomicAdd(&stats[5], n_steps);
        atomicAdd(&stats[6], n_lanes);
        atomicAdd(&stats[7], n_rounds);
    }
}

// Zeroes the work counter of the trace launch that follows (a launch that is not preceded by a sort).
__global__ void k_trace_arm(uint32_t *ctl, int wait) {
    if (wait) pdl_wait();
    pdl_trigger();
    if (threadIdx.x < 2) ctl[threadIdx.x] = 0u;
}

}  // namespace hcc

using namespace hcc;

// every launch takes the next counter slot of the ring, so launches in flight on different streams never share a
// counter (up to HCC_TRACE_SLOTS of them); the slot is zeroed on the launch stream by a kernel before the trace
// kernel (the sort's first kernel or k_trace_arm), so an aborted launch leaves nothing behind
uint32_t *hcc::trace_take_slot(const hcc_bvh *bvh) {
    return bvh->d_trace_ctl + 2u * (bvh->trace_calls->fetch_add(1u) % (uint32_t)HCC_TRACE_SLOTS);
}

int32_t hcc::trace_arm(uint32_t *slot, cudaStream_t s) {
    HCC_CUDA_TRY(launch_k(LK_FIRST, k_trace_arm, dim3(1), dim3(32), 0, s, slot, 1));
    return HCC_OK;
}

int32_t hcc::trace_launch(const char *who, const hcc_bvh *bvh, const float *rays_dev, uint64_t n, const uint32_t *perm_dev,
                          int32_t mode, void *hits_dev, unsigned long long *stats_dev, cudaStream_t s, uint32_t *armed_slot,
                          LaunchKind kind) {
    HCC_REQUIRE(bvh, HCC_ERR_INVALID_ARG, "%s: NULL bvh", who);
    HCC_REQUIRE(mode == HCC_TRACE_CLOSEST || mode == HCC_TRACE_ANY, HCC_ERR_INVALID_ARG, "%s: unknown mode %d", who, mode);
    if (n == 0) return HCC_OK;
    HCC_REQUIRE(rays_dev && hits_dev, HCC_ERR_INVALID_ARG, "%s: NULL argument", who);
    HCC_REQUIRE(aligned(rays_dev, 32) && aligned(hits_dev, 16) && aligned(perm_dev, 16), HCC_ERR_BAD_ALIGNMENT,
                "%s: rays need 32-byte, hits and perm 16-byte alignment", who);
    // the rank counter runs up to n + 32 * (warps of the grid) before every warp has seen it exhausted
    HCC_REQUIRE(n < (1ull << 32) - (1ull << 24), HCC_ERR_UNSUPPORTED, "%s: n >= 2^32 - 2^24", who);
    const uint32_t cap = (uint32_t)sm_count() * (mode == HCC_TRACE_ANY ? TRACE_BLOCKS_PER_SM_ANY : TRACE_BLOCKS_PER_SM);
    const uint32_t want = (uint32_t)((n + TRACE_THREADS - 1) / TRACE_THREADS);
    const uint32_t blocks = want < cap ? want : cap;
    TraceScene sc;
    sc.wrec = bvh->d_wrec; sc.ttri = bvh->d_ttri; sc.root_ref = bvh->root_ref;
    for (int a = 0; a < 3; ++a) { sc.q_lo[a] = bvh->q_lo[a]; sc.q_scale[a] = bvh->q_scale[a]; }
    // an armed slot: the trace kernel itself is launched as `kind`; else a one-warp kernel launched as `kind` arms a
    // fresh slot and the trace kernel is a chained launch behind it
    uint32_t *ctl = armed_slot;
    LaunchKind trace_kind = kind;
    if (!ctl) {
        ctl = trace_take_slot(bvh);
        HCC_CUDA_TRY(launch_k(kind, k_trace_arm, dim3(1), dim3(32), 0, s, ctl, kind_waits(kind)));
        trace_kind = LK_CHAIN;
    }
    sc.wait = (uint32_t)kind_waits(trace_kind);
    const float4 *rays = (const float4 *)rays_dev;
    const bool any = mode == HCC_TRACE_ANY;
#ifdef HCC_TRACE_TIMELINE   // debug builds: the plain kernel writes its per-warp times behind the counters
    auto kern = any ? k_trace<true, false> : k_trace<false, false>;
#else
    auto kern = stats_dev ? (any ? k_trace<true, true> : k_trace<false, true>) : (any ? k_trace<true, false> : k_trace<false, false>);
#endif
    HCC_CUDA_TRY(launch_k(trace_kind, kern, dim3(blocks), dim3(TRACE_THREADS), 0, s, sc, rays, perm_dev, (uint32_t)n, hits_dev, ctl, stats_dev));
    return HCC_OK;
}

extern "C" int32_t hcc_trace(const hcc_bvh *bvh, const float *rays_dev, uint64_t n, const uint32_t *perm_dev,
                             int32_t mode, void *hits_dev, void *stream) {
    return trace_launch("hcc_trace", bvh, rays_dev, n, perm_dev, mode, hits_dev, nullptr, (cudaStream_t)stream, nullptr, LK_FIRST);
}

extern "C" int32_t hcc_trace_stats(const hcc_bvh *bvh, const float *rays_dev, uint64_t n, const uint32_t *perm_dev,
                                   int32_t mode, void *hits_dev, uint64_t *stats_dev, void *stream) {
    HCC_REQUIRE(stats_dev && aligned(stats_dev, 16), HCC_ERR_INVALID_ARG, "hcc_trace_stats: stats_dev NULL or misaligned");
    HCC_CUDA_TRY(cudaMemsetAsync(stats_dev, 0, 8 * sizeof(uint64_t), (cudaStream_t)stream));
    return trace_launch("hcc_trace_stats", bvh, rays_dev, n, perm_dev, mode, hits_dev, (unsigned long long *)stats_dev, (cudaStream_t)stream, nullptr, LK_FIRST);
}
