// Shared host/device helpers of the CUDA path (sm_100a).  Nothing here is used by the
// oracle; the two share no code.
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>
#include <stdio.h>
#include <stdlib.h>

#include <atomic>

#include "../../include/hcc.h"

namespace hcc {

void set_error(const char *fmt, ...);

#define HCC_CUDA_TRY(expr)                                                              \
    do {                                                                                \
        cudaError_t _e = (expr);                                                        \
        if (_e != cudaSuccess) {                                                        \
            hcc::set_error("%s failed: %s (%s:%d)", #expr, cudaGetErrorString(_e),      \
                           __FILE__, __LINE__);                                         \
            return HCC_ERR_CUDA;                                                        \
        }                                                                               \
    } while (0)

#define HCC_REQUIRE(cond, status, ...)                                                  \
    do {                                                                                \
        if (!(cond)) {                                                                  \
            hcc::set_error(__VA_ARGS__);                                                \
            return (status);                                                            \
        }                                                                               \
    } while (0)

inline bool aligned(const void *p, uintptr_t a) { return (reinterpret_cast<uintptr_t>(p) & (a - 1)) == 0; }

constexpr int HCC_MAX_DEVICES = 64;
inline int current_device() {
    int dev = 0;
    if (cudaGetDevice(&dev) != cudaSuccess || dev < 0 || dev >= HCC_MAX_DEVICES) dev = 0;
    return dev;
}

// SM count of the current device (cached per device: one process may drive several)
inline int sm_count() {
    static std::atomic<int> n[HCC_MAX_DEVICES];
    const int dev = current_device();
    int v = n[dev].load(std::memory_order_relaxed);
    if (v == 0) {
        if (cudaDeviceGetAttribute(&v, cudaDevAttrMultiProcessorCount, dev) != cudaSuccess || v <= 0) v = 148;
        n[dev].store(v, std::memory_order_relaxed);
    }
    return v;
}

inline uint64_t round_up(uint64_t x, uint64_t a) { return (x + a - 1) / a * a; }

// ---- programmatic dependent launch (sm_90+).  The kernels of one library call form a chain: all but the
// first are launched with the programmatic-stream-serialization attribute, so a kernel may become resident
// while its predecessor still runs; it calls pdl_wait() before it touches anything a predecessor wrote (or
// may still read) and pdl_trigger() only AFTER that wait.  Rule of the chain: a kernel that is launched has
// seen its predecessor pass its own wait, so everything before the predecessor is complete; only the
// predecessor itself may still run.  The FIRST kernel of a call is a plain launch (LK_FIRST): ordered after
// everything enqueued on the stream before it.  LK_OVERLAP is for hcc_reorder_trace_pair only: the first
// kernel of the second batch's chain is a dependent launch that does NOT wait, so the chain runs while the
// first batch's traversal kernel drains.  HCC_NO_PDL=1 in the environment makes every launch a plain one.
enum LaunchKind { LK_FIRST = 0, LK_CHAIN = 1, LK_OVERLAP = 2 };

inline bool pdl_enabled() {
    static const bool on = [] { const char *e = getenv("HCC_NO_PDL"); return !(e && e[0] == '1'); }();
    return on;
}

template <typename... KArgs, typename... Args>
inline cudaError_t launch_k(LaunchKind kind, void (*kern)(KArgs...), dim3 grid, dim3 block, size_t smem, cudaStream_t s, Args... args) {
    cudaLaunchConfig_t cfg = {};
    cfg.gridDim = grid;
    cfg.blockDim = block;
    cfg.dynamicSmemBytes = smem;
    cfg.stream = s;
    cudaLaunchAttribute attr[1];
    attr[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
    attr[0].val.programmaticStreamSerializationAllowed = 1;
    cfg.attrs = attr;
    cfg.numAttrs = (kind != LK_FIRST && pdl_enabled()) ? 1 : 0;
    return cudaLaunchKernelEx(&cfg, kern, KArgs(args)...);
}
// does the first kernel of a chain launched as `kind` call pdl_wait()?  (a plain launch needs no wait, but the call is a
// no-op there; LK_OVERLAP must not wait - unless dependent launches are off, then it is a plain launch anyway)
inline int kind_waits(LaunchKind kind) { return kind == LK_OVERLAP ? 0 : 1; }

#ifdef __CUDACC__
__device__ __forceinline__ void pdl_wait() { asm volatile("griddepcontrol.wait;" ::: "memory"); }
__device__ __forceinline__ void pdl_trigger() { asm volatile("griddepcontrol.launch_dependents;" ::: "memory"); }
#endif

// Traversal grid (bvh.cu, trace.cu): child boxes are stored as 15-bit cell indices of a
// uniform grid over the root box, rounded outwards and padded by one cell.
constexpr float HCC_GRID_CELLS = 32763.0f;
constexpr float HCC_GRID_OFFSET = 2.0f;
constexpr uint32_t HCC_REF_LEAF = 0x80000000u;
// Extra slack of the traversal's slab test, as a fraction of (|ray origin in cells| + 65536): 2^-20,
// about four times the rounding of the fp32 plane distances (trace.cu).
constexpr float HCC_TRACE_PAD = 9.5367431640625e-07f;
constexpr int HCC_TRACE_SLOTS = 1024;   // work counters of trace launches in flight on one BVH

// Device-side level tables of a cut hierarchy, passed to kernels by value.
struct CutDev {
    uint32_t m;                        // number of levels
    uint32_t w[HCC_MAX_LEVELS];        // level widths
    uint32_t ent_off[HCC_MAX_LEVELS];  // first entry of level l in the flat arrays
    uint32_t tab_off[HCC_MAX_LEVELS];  // first table of level l
    uint32_t n_tab[HCC_MAX_LEVELS];    // tables on level l = prod(w[0..l-1])
    uint32_t n_entries;                // sum over levels of n_tab*w
    uint32_t n_tables;
    uint32_t bits_used;
    const float4 *boxes;               // 2 float4 per entry: (lo.x, lo.y, hi.x, hi.y), (lo.z, hi.z, cnt-of-table in entry 0, -)
    const uint32_t *entry_node;
    const uint32_t *table_cnt;
};

}  // namespace hcc

struct hcc_bvh {
    uint32_t n_nodes, n_tris, n_leaves, max_depth;
    float scene_lo[3], scene_hi[3];
    hcc_node *d_nodes;      // canonical nodes
    uint32_t *d_parent;     // parent index (root: 0xFFFFFFFF)
    uint32_t *d_leaves;     // sub-tree leaf counts
    uint32_t *d_flags;      // arrival counters of the bottom-up passes
    uint32_t *d_internal;   // indices of the internal nodes, ascending
    uint32_t *d_wrec;       // traversal records: 16 words (64 bytes) per node of the 4-wide tree (bvh.cu)
    uint32_t n_wide;
    float4 *d_ttri;         // 4 float4 (64 bytes) per triangle, leaf order
    uint32_t n_internal;
    uint32_t root_ref;      // traversal reference of the root (see bvh.cu)
    uint32_t *d_trace_ctl;  // HCC_TRACE_SLOTS x {next rank, -}: work counters of trace launches in flight
    std::atomic<uint32_t> *trace_calls;
    float q_lo[3], q_scale[3];   // traversal grid: g = (x - q_lo) * q_scale + HCC_GRID_OFFSET
    // scratch for hcc_select_cut_flat lives in the caller's workspace
};

struct hcc_cut {
    uint32_t cap_entries, cap_tables;
    uint32_t K_eff, key_bits, container_bits;
    uint32_t flags;         // HCC_CUT_* of the last selection
    hcc::CutDev dev;        // pointers into the buffers below
    float4 *d_boxes;
    uint32_t *d_entry_node;
    uint32_t *d_table_cnt;
    bool valid;
};

// stage entry points implemented in the other translation units
namespace hcc {
int32_t launch_build_tables(const hcc_bvh *bvh, const float *had, hcc_cut *cut, cudaStream_t s);
// The hot-path stages as hcc_reorder_trace chains them; `kind` is how the stage's first kernel is launched.
int32_t encode_launch(const float *rays_dev, uint64_t n, const hcc_cut *cut, void *keys_dev, cudaStream_t s, LaunchKind kind);
int32_t encode_twopoint_launch(const float *rays_dev, uint64_t n, const float scene_lo[3], const float scene_hi[3],
                               uint32_t key_bits, void *keys_dev, cudaStream_t s, LaunchKind kind);
// also_zero: two words the sort's first kernel zeroes besides its own control region (the trace work counter), or NULL
int32_t sort_launch(void *keys_dev, uint64_t n, uint32_t container_bits, uint32_t bit_lo, uint32_t bit_hi, uint32_t *perm_dev,
                    void *workspace_dev, uint64_t workspace_bytes, cudaStream_t s, uint32_t *also_zero, LaunchKind kind);
uint32_t *trace_take_slot(const hcc_bvh *bvh);
int32_t trace_arm(uint32_t *slot, cudaStream_t s);      // zero a work counter by a plain one-warp launch
// armed_slot: a work counter already zeroed by an earlier kernel: the trace kernel itself is launched as `kind`; or
// NULL: a one-warp kernel launched as `kind` zeroes a fresh counter and the trace kernel is a chained launch behind it
int32_t trace_launch(const char *who, const hcc_bvh *bvh, const float *rays_dev, uint64_t n, const uint32_t *perm_dev, int32_t mode,
                     void *hits_dev, unsigned long long *stats_dev, cudaStream_t s, uint32_t *armed_slot, LaunchKind kind);
}
