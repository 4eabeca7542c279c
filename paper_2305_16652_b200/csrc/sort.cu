// (a3) sort of (key, ray id) pairs: stable LSD radix sort, 8-bit digits, one chained-scan
// ("onesweep") kernel per digit with warp match ranking and decoupled look-back.
// PAPER.md:196 ("sorting the HCCs as natural numbers"), :247 ("sorts the indices of rays").
// The paper calls Thrust; this is a from-scratch sm_100a kernel family.
#include "common.cuh"

namespace hcc {

constexpr int RADIX_BITS = 8;
constexpr int RADIX = 1 << RADIX_BITS;
// Tile shape (4096 pairs per CTA): 256 threads x 16 pairs for both key widths (overridable at build
// time for tuning); launch bounds cap the registers at 4 (32-bit keys) resp. 3 (64-bit keys) CTAs
// per SM because occupancy, not bandwidth, decides this kernel's speed.
#ifndef HCC_SORT32_THREADS
#define HCC_SORT32_THREADS 256
#define HCC_SORT32_ITEMS 16
#define HCC_SORT32_MIN_CTAS 4
#endif
#ifndef HCC_SORT64_THREADS
#define HCC_SORT64_THREADS 256
#define HCC_SORT64_ITEMS 16
#define HCC_SORT64_MIN_CTAS 3
#endif
template <typename KeyT> struct SortCfg {
    static constexpr int THREADS = HCC_SORT32_THREADS, ITEMS = HCC_SORT32_ITEMS, MIN_CTAS = HCC_SORT32_MIN_CTAS;
};
template <> struct SortCfg<unsigned long long> {
    static constexpr int THREADS = HCC_SORT64_THREADS, ITEMS = HCC_SORT64_ITEMS, MIN_CTAS = HCC_SORT64_MIN_CTAS;
};
constexpr int SORT_TILE = HCC_SORT32_THREADS * HCC_SORT32_ITEMS;
static_assert(HCC_SORT64_THREADS * HCC_SORT64_ITEMS == SORT_TILE, "both key widths use the same tile size");
constexpr int MAX_PASSES = 8;
constexpr uint32_t FLAG_AGG = 1u << 30, FLAG_PREFIX = 2u << 30, VAL_MASK = (1u << 30) - 1u;
constexpr int HIST_THREADS = 256;
#ifndef HCC_HIST_BATCH
#define HCC_HIST_BATCH 4
#endif
constexpr int HIST_BATCH = HCC_HIST_BATCH;
#ifndef HCC_SORT_FEW
#define HCC_SORT_FEW 20
#endif
constexpr float MATCH_MAX_DISTINCT = (float)HCC_SORT_FEW;   // expected distinct digits per warp up to which MATCH.ANY is used
constexpr int LOOK = 4;                      // look-back rows fetched per round trip

// control region of the workspace (zeroed at the start of every sort by k_sort_init, the first kernel of its chain)
struct SortCtl {
    uint32_t hist[MAX_PASSES][RADIX];
    uint32_t ticket[MAX_PASSES];
    uint32_t few_digits[MAX_PASSES];   // pass p: a warp's 32 keys are expected to hold few distinct digits

};

__device__ __forceinline__ uint32_t ld_volatile_u32(const uint32_t *p) {
    uint32_t v;
    asm volatile("ld.volatile.global.u32 %0, [%1];" : "=r"(v) : "l"(p));
    return v;
}
__device__ __forceinline__ void st_volatile_u32(uint32_t *p, uint32_t v) {
    asm volatile("st.volatile.global.u32 [%0], %1;" ::"l"(p), "r"(v) : "memory");
}

// First kernel of a sort: zeroes the control region and the status rows of the passes (uint4 stores) and, for
// hcc_reorder_trace, the work counter of the trace launch that follows the sort.
__global__ void __launch_bounds__(256) k_sort_init(uint4 *__restrict__ zero, size_t n_vec, uint32_t *also_zero, int wait) {
    if (wait) pdl_wait();
    pdl_trigger();
    const size_t stride = (size_t)gridDim.x * blockDim.x;
    for (size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x; i < n_vec; i += stride) zero[i] = make_uint4(0u, 0u, 0u, 0u);
    if (also_zero && blockIdx.x == 0 && threadIdx.x < 2) also_zero[threadIdx.x] = 0u;
}

// All digit histograms in one read of the keys.
template <typename KeyT>
__global__ void __launch_bounds__(HIST_THREADS)
k_histogram(const KeyT *__restrict__ keys, uint32_t n, uint32_t passes, uint32_t bit_lo, SortCtl *ctl) {
    __shared__ uint32_t sh[MAX_PASSES][RADIX];
    for (uint32_t i = threadIdx.x; i < MAX_PASSES * RADIX; i += HIST_THREADS) (&sh[0][0])[i] = 0u;
    pdl_wait();
    pdl_trigger();
    __syncthreads();
    // 16 bytes of keys per load and HIST_BATCH independent loads in flight per thread: the kernel is
    // a pure stream and would otherwise wait one DRAM round trip per key
    constexpr uint32_t PER = 16 / sizeof(KeyT);
    const uint32_t n_vec = n / PER;
    const uint4 *vec = reinterpret_cast<const uint4 *>(keys);
    const uint32_t stride = gridDim.x * HIST_THREADS;
    auto count = [&](KeyT k) {
        for (uint32_t p = 0; p < passes; ++p) atomicAdd(&sh[p][(uint32_t)(k >> (bit_lo + RADIX_BITS * p)) & (RADIX - 1)], 1u);
    };
    for (uint32_t i = blockIdx.x * HIST_THREADS + threadIdx.x; i < n_vec; i += HIST_BATCH * stride) {
        uint4 v[HIST_BATCH];
#pragma unroll
        for (int b = 0; b < HIST_BATCH; ++b) {
            const uint32_t j = i + b * stride;
            v[b] = j < n_vec ? vec[j] : make_uint4(0u, 0u, 0u, 0u);
        }
#pragma unroll
        for (int b = 0; b < HIST_BATCH; ++b) {
            if (i + b * stride < n_vec) {
                if (sizeof(KeyT) == 4) { count((KeyT)v[b].x); count((KeyT)v[b].y); count((KeyT)v[b].z); count((KeyT)v[b].w); }
                else { count((KeyT)(((unsigned long long)v[b].y << 32) | v[b].x)); count((KeyT)(((unsigned long long)v[b].w << 32) | v[b].z)); }
            }
        }
    }
    for (uint32_t i = n_vec * PER + blockIdx.x * HIST_THREADS + threadIdx.x; i < n; i += stride) count(keys[i]);   // ragged tail
    __syncthreads();
    for (uint32_t i = threadIdx.x; i < passes * RADIX; i += HIST_THREADS) {
        uint32_t c = (&sh[0][0])[i];
        if (c) atomicAdd(&(&ctl->hist[0][0])[i], c);
    }
}

// Exclusive scan of each digit histogram, written as the PREFIX row of "tile -1"
// (row 0 of that pass's status array), so the look-back needs no special first tile.
__global__ void __launch_bounds__(RADIX)
k_scan_hist(SortCtl *ctl, uint32_t *status, size_t status_stride, uint32_t n) {
    __shared__ uint32_t s_w[RADIX / 32];
    __shared__ float s_e[RADIX / 32];
    const uint32_t p = blockIdx.x, d = threadIdx.x, lane = d & 31u, warp = d >> 5;
    pdl_wait();
    pdl_trigger();
    uint32_t v = ctl->hist[p][d], incl = v;
#pragma unroll
    for (int o = 1; o < 32; o <<= 1) {
        uint32_t x = __shfl_up_sync(0xFFFFFFFFu, incl, o);
        if (lane >= (uint32_t)o) incl += x;
    }
    if (lane == 31) s_w[warp] = incl;
    // expected number of distinct digits among the 32 keys of a warp = sum_d 1 - (1 - p_d)^32:
    // MATCH.ANY costs a round per distinct value, the ballot form a fixed 9 rounds
    float e = v ? 1.0f - exp2f(32.0f * log2f(fmaxf(1.0f - (float)v / (float)n, 1e-30f))) : 0.0f;
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) e += __shfl_xor_sync(0xFFFFFFFFu, e, o);
    if (lane == 0) s_e[warp] = e;
    __syncthreads();
    if (d == 0) {
        float tot = 0.0f;
        for (int w = 0; w < RADIX / 32; ++w) tot += s_e[w];
        ctl->few_digits[p] = tot <= MATCH_MAX_DISTINCT ? 1u : 0u;
    }
    uint32_t add = 0;
    for (uint32_t w = 0; w < warp; ++w) add += s_w[w];
    status[p * status_stride + d] = FLAG_PREFIX | (add + incl - v);
}

__global__ void k_iota(uint32_t *perm, uint32_t n) {
    uint32_t i = blockIdx.x * blockDim.x + threadIdx.x;
    pdl_wait();
    pdl_trigger();
    if (i < n) perm[i] = i;
}

// One radix pass.  status: (tiles + 1) rows of RADIX words for this pass; row t+1 belongs to
// tile t: empty (0), AGG | count of the tile, or PREFIX | count of tiles 0..t plus the digit's
// global base.  Tiles are handed out by an atomic ticket so that every predecessor of a
// running tile is itself running or done (forward progress of the look-back spin).
template <typename KeyT, bool FIRST, bool WRITE_KEYS>
__global__ void __launch_bounds__(SortCfg<KeyT>::THREADS, SortCfg<KeyT>::MIN_CTAS)
k_onesweep(const KeyT *__restrict__ keys_in, KeyT *__restrict__ keys_out, const uint32_t *__restrict__ vals_in,
           uint32_t *__restrict__ vals_out, uint32_t n, uint32_t shift, uint32_t *status, uint32_t *ticket,
           const uint32_t *few_digits, uint32_t tiles) {
    constexpr int SORT_THREADS = SortCfg<KeyT>::THREADS, SORT_ITEMS = SortCfg<KeyT>::ITEMS, SORT_WARPS = SORT_THREADS / 32;
    static_assert(SORT_THREADS * SORT_ITEMS == SORT_TILE && SORT_THREADS >= RADIX, "tile shape");
    __shared__ uint32_t s_warp_hist[SORT_WARPS][RADIX];
    __shared__ uint32_t s_tile_off[RADIX];
    __shared__ uint32_t s_gbase[RADIX];
    __shared__ uint32_t s_warp_tot[RADIX / 32];
    __shared__ uint32_t s_ticket[2];
    extern __shared__ __align__(16) unsigned char s_dyn[];
    KeyT *s_keys = reinterpret_cast<KeyT *>(s_dyn);
    uint32_t *s_vals = reinterpret_cast<uint32_t *>(s_dyn + sizeof(KeyT) * SORT_TILE);

    const uint32_t tid = threadIdx.x, lane = tid & 31u, warp = tid >> 5;
    pdl_wait();          // the previous pass (or the histogram scan) is complete
    pdl_trigger();
    const bool use_match = *few_digits != 0u;      // uniform over the grid
    const uint32_t my_base = warp * (SORT_ITEMS * 32) + lane;   // item i at my_base + 32*i (warp-striped)
    KeyT key[SORT_ITEMS];
    uint32_t rank[SORT_ITEMS];
    auto load_keys = [&](uint32_t t) {
        const uint32_t base = t * SORT_TILE, cnt = min((uint32_t)SORT_TILE, n - base);
#pragma unroll
        for (int i = 0; i < SORT_ITEMS; ++i) {
            const uint32_t idx = my_base + 32 * i;
            key[i] = idx < cnt ? keys_in[base + idx] : (KeyT)0;
        }
    };
    // 64-bit keys also bring the next tile's ray ids in early (the 32-bit kernel has no registers to spare)
    constexpr bool PREFETCH_VALS = !FIRST && sizeof(KeyT) == 8;
    uint32_t val[PREFETCH_VALS ? SORT_ITEMS : 1];
    auto load_vals = [&](uint32_t t) {
        const uint32_t base = t * SORT_TILE, cnt = min((uint32_t)SORT_TILE, n - base);
#pragma unroll
        for (int i = 0; i < SORT_ITEMS; ++i) {
            const uint32_t idx = my_base + 32 * i;
            val[PREFETCH_VALS ? i : 0] = idx < cnt ? vals_in[base + idx] : 0u;
        }
    };
    if (tid == 0) s_ticket[0] = atomicAdd(ticket, 1u);
    __syncthreads();
    uint32_t tile = s_ticket[0], slot = 0;
    if (tile < tiles) {
        load_keys(tile);
        if (PREFETCH_VALS) load_vals(tile);
    }
  while (tile < tiles) {                           // persistent: one CTA works through many tiles
    for (uint32_t i = tid; i < SORT_WARPS * RADIX; i += SORT_THREADS) (&s_warp_hist[0][0])[i] = 0u;
    if (tid == 0) s_ticket[slot ^ 1u] = atomicAdd(ticket, 1u);
    __syncthreads();
    const uint32_t next = s_ticket[slot ^ 1u];
    const uint32_t tile_base = tile * SORT_TILE;
    const uint32_t count = min((uint32_t)SORT_TILE, n - tile_base);

    // rank every item among the equal digits of its warp, in (item, lane) order
    const uint32_t lt = (1u << lane) - 1u;
#pragma unroll
    for (int i = 0; i < SORT_ITEMS; ++i) {
        const bool valid = my_base + 32 * i < count;
        const uint32_t digit = valid ? ((uint32_t)(key[i] >> shift) & (RADIX - 1)) : (uint32_t)RADIX;
        // lanes holding the same digit.  MATCH.ANY costs a round per distinct value in the warp:
        // it wins when the pass has few distinct digits (hierarchy cut codes are like that), one
        // ballot per digit bit wins on well-spread digits (TwoPoint's Morton codes)
        uint32_t peers;
        if (use_match) {
            peers = __match_any_sync(0xFFFFFFFFu, digit);
        } else {
            peers = 0xFFFFFFFFu;
#pragma unroll
            for (int b = 0; b <= RADIX_BITS; ++b) {
                const bool bit = (digit >> b) & 1u;
                const uint32_t m = __ballot_sync(0xFFFFFFFFu, bit);
                peers &= bit ? m : ~m;
            }
        }
        const uint32_t below = __popc(peers & lt);
        const uint32_t old = s_warp_hist[warp][digit & (RADIX - 1)];
        __syncwarp();
        if (valid && below == 0) s_warp_hist[warp][digit] = old + __popc(peers);
        __syncwarp();
        rank[i] = old + below;
    }
    __syncthreads();

    // thread d: digit d.  Warp-exclusive offsets, tile total, publish the aggregate, scan over digits.
    const uint32_t d = tid;
    uint32_t total = 0, excl_local = 0, incl = 0;
    uint32_t *row = status + (size_t)(tile + 1) * RADIX;
    if (d < RADIX) {
        uint32_t run = 0;
#pragma unroll
        for (int w = 0; w < SORT_WARPS; ++w) {
            uint32_t t = s_warp_hist[w][d];
            s_warp_hist[w][d] = run;
            run += t;
        }
        total = run;
        st_volatile_u32(row + d, FLAG_AGG | total);
        incl = total;
#pragma unroll
        for (int o = 1; o < 32; o <<= 1) {
            uint32_t x = __shfl_up_sync(0xFFFFFFFFu, incl, o);
            if (lane >= (uint32_t)o) incl += x;
        }
        if (lane == 31) s_warp_tot[warp] = incl;
    }
    __syncthreads();
    if (d < RADIX) {
        uint32_t add = 0;
        for (uint32_t w = 0; w < warp; ++w) add += s_warp_tot[w];
        excl_local = add + incl - total;
        s_tile_off[d] = excl_local;
    }
    __syncthreads();

    // scatter into tile order in shared memory: needs the tile-local offsets only, so it runs
    // BEFORE the look-back and gives the predecessors time to publish
#pragma unroll
    for (int i = 0; i < SORT_ITEMS; ++i) {
        const uint32_t idx = my_base + 32 * i;
        if (idx < count) {
            const uint32_t digit = (uint32_t)(key[i] >> shift) & (RADIX - 1);
            const uint32_t p = s_tile_off[digit] + s_warp_hist[warp][digit] + rank[i];
            s_keys[p] = key[i];
            s_vals[p] = FIRST ? tile_base + idx : (PREFETCH_VALS ? val[PREFETCH_VALS ? i : 0] : vals_in[tile_base + idx]);
        }
    }

    // the key registers are free now: bring in the next tile's keys while this tile looks back and
    // writes out
    if (next < tiles) {
        load_keys(next);
        if (PREFETCH_VALS) load_vals(next);
    }

    // decoupled look-back over rows tile, tile-1, ..., 0 (row 0 = seeded global digit base).
    // LOOK rows are read at once: a walk over aggregates costs one L2 round trip per LOOK rows
    // instead of one per row.  Rows before row 0 are never reached logically (row 0 is a
    // PREFIX); the speculative reads of them stay inside the workspace.
    if (d < RADIX) {
        uint32_t excl = 0;
        const uint32_t *prow = status + (size_t)tile * RADIX + d;
        for (bool done = false; !done;) {
            uint32_t v[LOOK];
#pragma unroll
            for (int k = 0; k < LOOK; ++k) v[k] = ld_volatile_u32(prow - (ptrdiff_t)k * RADIX);
            int k = 0;
#pragma unroll
            for (; k < LOOK; ++k) {
                if ((v[k] >> 30) == 0u) break;
                excl += v[k] & VAL_MASK;
                if (v[k] & FLAG_PREFIX) { done = true; break; }
            }
            prow -= (ptrdiff_t)k * RADIX;
        }
        st_volatile_u32(row + d, FLAG_PREFIX | ((excl + total) & VAL_MASK));
        s_gbase[d] = excl - excl_local;
    }
    __syncthreads();
    // write out: consecutive threads -> consecutive addresses inside each digit run
    for (uint32_t p = tid; p < count; p += SORT_THREADS) {
        const KeyT k = s_keys[p];
        const uint32_t pos = s_gbase[(uint32_t)(k >> shift) & (RADIX - 1)] + p;
        if (WRITE_KEYS) keys_out[pos] = k;
        vals_out[pos] = s_vals[p];
    }
    __syncthreads();                               // shared buffers and the ticket slot are reused by the next tile
    tile = next;
    slot ^= 1u;
  }
}

static uint64_t ctl_bytes(uint64_t n) {
    uint64_t tiles = (n + SORT_TILE - 1) / SORT_TILE;
    return round_up(sizeof(SortCtl), 256) + round_up((uint64_t)MAX_PASSES * (tiles + 1) * RADIX * sizeof(uint32_t), 256);
}

template <typename KeyT>
static int32_t sort_impl(KeyT *keys, uint32_t n, uint32_t passes, uint32_t bit_lo, uint32_t *perm, unsigned char *ws, cudaStream_t s, uint32_t *also_zero, LaunchKind kind) {
    const uint32_t tiles = (n + SORT_TILE - 1) / SORT_TILE;
    KeyT *keys_tmp = reinterpret_cast<KeyT *>(ws);
    uint32_t *vals_tmp = reinterpret_cast<uint32_t *>(ws + round_up(sizeof(KeyT) * (uint64_t)n, 256));
    unsigned char *ctl_raw = ws + round_up(sizeof(KeyT) * (uint64_t)n, 256) + round_up(sizeof(uint32_t) * (uint64_t)n, 256);
    SortCtl *ctl = reinterpret_cast<SortCtl *>(ctl_raw);
    uint32_t *status = reinterpret_cast<uint32_t *>(ctl_raw + round_up(sizeof(SortCtl), 256));
    const size_t status_stride = (size_t)(tiles + 1) * RADIX;
    {
        const size_t zero_bytes = round_up(sizeof(SortCtl), 256) + (size_t)passes * status_stride * sizeof(uint32_t);   // a multiple of 16
        const size_t n_vec = zero_bytes / 16;
        size_t blocks = (n_vec + 256 * 8 - 1) / (256 * 8);
        const size_t cap_init = (size_t)sm_count() * 8;
        if (blocks > cap_init) blocks = cap_init;
        HCC_CUDA_TRY(launch_k(kind, k_sort_init, dim3((unsigned)blocks), dim3(256), 0, s, reinterpret_cast<uint4 *>(ctl_raw), n_vec, also_zero, kind_waits(kind)));
    }
    int hist_blocks = (int)((n + HIST_THREADS * 16 - 1) / (HIST_THREADS * 16));
    int cap = sm_count() * 8;
    if (hist_blocks > cap) hist_blocks = cap;
    HCC_CUDA_TRY(launch_k(LK_CHAIN, k_histogram<KeyT>, dim3(hist_blocks), dim3(HIST_THREADS), 0, s, (const KeyT *)keys, n, passes, bit_lo, ctl));
    HCC_CUDA_TRY(launch_k(LK_CHAIN, k_scan_hist, dim3(passes), dim3(RADIX), 0, s, ctl, status, status_stride, n));
    const size_t dyn = (sizeof(KeyT) + sizeof(uint32_t)) * SORT_TILE;
    constexpr int SORT_THREADS = SortCfg<KeyT>::THREADS;
    // once per device and key width: the dynamic shared-memory limit and the resident CTAs per SM
    static std::atomic<int> per_sm_cache[HCC_MAX_DEVICES];
    const int dev = current_device();
    int per_sm = per_sm_cache[dev].load(std::memory_order_acquire);
    if (per_sm == 0) {
        HCC_CUDA_TRY(cudaFuncSetAttribute(k_onesweep<KeyT, true, true>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)dyn));
        HCC_CUDA_TRY(cudaFuncSetAttribute(k_onesweep<KeyT, true, false>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)dyn));
        HCC_CUDA_TRY(cudaFuncSetAttribute(k_onesweep<KeyT, false, true>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)dyn));
        HCC_CUDA_TRY(cudaFuncSetAttribute(k_onesweep<KeyT, false, false>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)dyn));
        if (cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, k_onesweep<KeyT, false, true>, SORT_THREADS, dyn) != cudaSuccess || per_sm < 1) per_sm = 1;
        per_sm_cache[dev].store(per_sm, std::memory_order_release);
    }
    const uint32_t resident = (uint32_t)(sm_count() * per_sm);
    const uint32_t grid = tiles < resident ? tiles : resident;     // every CTA resident: the look-back cannot starve
    KeyT *kin = keys, *kout = keys_tmp;
    for (uint32_t p = 0; p < passes; ++p) {
        const bool first = p == 0, last = p + 1 == passes;
        // the last pass must land in perm; value buffers alternate backwards from there
        uint32_t *vout = ((passes - 1 - p) & 1u) ? vals_tmp : perm;
        uint32_t *vin = ((passes - 1 - p) & 1u) ? perm : vals_tmp;
        uint32_t *st = status + (size_t)p * status_stride;
        uint32_t *tk = &ctl->ticket[p];
        const uint32_t *fd = &ctl->few_digits[p];
        const uint32_t shift = bit_lo + RADIX_BITS * p;
        auto kern = first && last ? k_onesweep<KeyT, true, false> : first ? k_onesweep<KeyT, true, true>
                    : last ? k_onesweep<KeyT, false, false> : k_onesweep<KeyT, false, true>;
        HCC_CUDA_TRY(launch_k(LK_CHAIN, kern, dim3(grid), dim3(SORT_THREADS), dyn, s, (const KeyT *)kin, kout, (const uint32_t *)vin, vout, n, shift, st, tk, fd, tiles));
        KeyT *t = kin; kin = kout; kout = t;
    }
    HCC_CUDA_TRY(cudaGetLastError());
    return HCC_OK;
}

}  // namespace hcc

using namespace hcc;

extern "C" int32_t hcc_sort_workspace_bytes(uint64_t n, uint32_t container_bits, uint64_t *bytes) {
    HCC_REQUIRE(bytes, HCC_ERR_INVALID_ARG, "hcc_sort_workspace_bytes: NULL bytes");
    HCC_REQUIRE(container_bits == 32 || container_bits == 64, HCC_ERR_INVALID_ARG, "hcc_sort: container_bits must be 32 or 64");
    HCC_REQUIRE(n < (1ull << 30), HCC_ERR_UNSUPPORTED, "hcc_sort: n >= 2^30");
    *bytes = round_up((container_bits / 8) * n, 256) + round_up(4 * n, 256) + ctl_bytes(n) + 256;
    return HCC_OK;
}

int32_t hcc::sort_launch(void *keys_dev, uint64_t n, uint32_t container_bits, uint32_t bit_lo, uint32_t bit_hi, uint32_t *perm_dev,
                         void *workspace_dev, uint64_t workspace_bytes, cudaStream_t s, uint32_t *also_zero, LaunchKind kind) {
    HCC_REQUIRE(container_bits == 32 || container_bits == 64, HCC_ERR_INVALID_ARG, "hcc_sort: container_bits must be 32 or 64");
    HCC_REQUIRE(bit_lo <= bit_hi && bit_hi <= container_bits, HCC_ERR_INVALID_ARG, "hcc_sort: need bit_lo <= bit_hi <= container_bits");
    HCC_REQUIRE(n < (1ull << 30), HCC_ERR_UNSUPPORTED, "hcc_sort: n >= 2^30");
    if (n == 0) return HCC_OK;
    HCC_REQUIRE(keys_dev && perm_dev && workspace_dev, HCC_ERR_INVALID_ARG, "hcc_sort: NULL argument");
    HCC_REQUIRE(aligned(keys_dev, 16) && aligned(perm_dev, 16) && aligned(workspace_dev, 16), HCC_ERR_BAD_ALIGNMENT,
                "hcc_sort: keys, perm and workspace need 16-byte alignment");
    uint64_t need = 0;
    hcc_sort_workspace_bytes(n, container_bits, &need);
    HCC_REQUIRE(workspace_bytes >= need, HCC_ERR_INVALID_ARG, "hcc_sort: workspace too small (%llu < %llu)",
                (unsigned long long)workspace_bytes, (unsigned long long)need);
    const uint32_t passes = (bit_hi - bit_lo + RADIX_BITS - 1) / RADIX_BITS;
    unsigned char *ws = reinterpret_cast<unsigned char *>(round_up(reinterpret_cast<uintptr_t>(workspace_dev), 256));
    if (passes == 0) {
        HCC_CUDA_TRY(launch_k(kind, k_sort_init, dim3(1), dim3(256), 0, s, reinterpret_cast<uint4 *>(ws), (size_t)0, also_zero, kind_waits(kind)));
        HCC_CUDA_TRY(launch_k(LK_CHAIN, k_iota, dim3((uint32_t)((n + 255) / 256)), dim3(256), 0, s, perm_dev, (uint32_t)n));
        return HCC_OK;
    }
    if (container_bits == 32) return sort_impl<uint32_t>((uint32_t *)keys_dev, (uint32_t)n, passes, bit_lo, perm_dev, ws, s, also_zero, kind);
    return sort_impl<unsigned long long>((unsigned long long *)keys_dev, (uint32_t)n, passes, bit_lo, perm_dev, ws, s, also_zero, kind);
}

extern "C" int32_t hcc_sort_range(void *keys_dev, uint64_t n, uint32_t container_bits, uint32_t bit_lo, uint32_t bit_hi,
                                  uint32_t *perm_dev, void *workspace_dev, uint64_t workspace_bytes, void *stream) {
    return sort_launch(keys_dev, n, container_bits, bit_lo, bit_hi, perm_dev, workspace_dev, workspace_bytes, (cudaStream_t)stream, nullptr, LK_FIRST);
}

extern "C" int32_t hcc_sort(void *keys_dev, uint64_t n, uint32_t container_bits, uint32_t bits_used, uint32_t *perm_dev,
                            void *workspace_dev, uint64_t workspace_bytes, void *stream) {
    HCC_REQUIRE(bits_used <= container_bits, HCC_ERR_INVALID_ARG, "hcc_sort: bits_used > container_bits");
    return hcc_sort_range(keys_dev, n, container_bits, 0u, bits_used, perm_dev, workspace_dev, workspace_bytes, stream);
}

// ---- hcc_sort_static: the sort for callers that cannot allocate device memory (include/hcc.h) ----------------
// The workspace is this array.  It is part of the library image: each GPU that loads these kernels holds it
// until the process exits.  On the host the name `g_sort_static_ws` is only a handle for the runtime, not a
// device address, so host code never passes it to a kernel: the address comes from cudaGetSymbolAddress, asked
// once per device with that device current.
static __device__ __align__(256) unsigned char g_sort_static_ws[HCC_SORT_STATIC_BYTES];

namespace {
constexpr uint64_t up256(uint64_t x) { return (x + 255u) / 256u * 256u; }
// hcc_sort_workspace_bytes(HCC_SORT_STATIC_MAX_N, 64) written out as a constant expression (64-bit keys need the most)
constexpr uint64_t STATIC_TILES = ((uint64_t)HCC_SORT_STATIC_MAX_N + hcc::SORT_TILE - 1) / hcc::SORT_TILE;
constexpr uint64_t STATIC_NEED = up256(8ull * HCC_SORT_STATIC_MAX_N) + up256(4ull * HCC_SORT_STATIC_MAX_N) + up256(sizeof(hcc::SortCtl)) +
                                 up256((uint64_t)hcc::MAX_PASSES * (STATIC_TILES + 1) * hcc::RADIX * sizeof(uint32_t)) + 256;
static_assert(STATIC_NEED <= HCC_SORT_STATIC_BYTES, "HCC_SORT_STATIC_BYTES too small for HCC_SORT_STATIC_MAX_N pairs");

// device address of g_sort_static_ws on the current device (looked up on the first call there, then cached)
int32_t static_ws(unsigned char **out) {
    static std::atomic<unsigned char *> cache[HCC_MAX_DEVICES];
    int dev = -1;
    HCC_CUDA_TRY(cudaGetDevice(&dev));
    HCC_REQUIRE(dev >= 0 && dev < HCC_MAX_DEVICES, HCC_ERR_UNSUPPORTED, "hcc_sort_static: device ordinal %d not supported", dev);
    unsigned char *p = cache[dev].load(std::memory_order_acquire);
    if (!p) {
        void *sym = nullptr;
        HCC_CUDA_TRY(cudaGetSymbolAddress(&sym, g_sort_static_ws));
        HCC_REQUIRE(sym && aligned(sym, 256), HCC_ERR_CUDA, "hcc_sort_static: no device address for the static workspace");
        p = static_cast<unsigned char *>(sym);
        cache[dev].store(p, std::memory_order_release);
    }
    *out = p;
    return HCC_OK;
}
}  // namespace

extern "C" int32_t hcc_sort_static(void *keys_dev, uint64_t n, uint32_t container_bits, uint32_t bits_used, uint32_t *perm_dev,
                                   void *stream) {
    HCC_REQUIRE(container_bits == 32 || container_bits == 64, HCC_ERR_INVALID_ARG, "hcc_sort_static: container_bits must be 32 or 64");
    HCC_REQUIRE(bits_used <= container_bits, HCC_ERR_INVALID_ARG, "hcc_sort_static: bits_used > container_bits");
    HCC_REQUIRE(n <= HCC_SORT_STATIC_MAX_N, HCC_ERR_UNSUPPORTED,
                "hcc_sort_static: n = %llu exceeds the static workspace's limit of %u pairs (use hcc_sort with a workspace of your own)",
                (unsigned long long)n, (unsigned)HCC_SORT_STATIC_MAX_N);
    if (n == 0) return HCC_OK;
    unsigned char *ws = nullptr;
    const int32_t rc = static_ws(&ws);
    if (rc != HCC_OK) return rc;
    // the same kernels as hcc_sort; k_sort_init, the first of them, zeroes the control region the last call left behind
    return sort_launch(keys_dev, n, container_bits, 0u, bits_used, perm_dev, ws, HCC_SORT_STATIC_BYTES, (cudaStream_t)stream, nullptr, LK_FIRST);
}
