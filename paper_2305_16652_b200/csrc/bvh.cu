// BVH upload + GPU layout conversion, and (a1) hierarchically accumulated density
// (Eq. 1 at :187).  Compiled with -fmad=false: every source-level
// floating-point operation is one IEEE fp32 operation.
#include <stdarg.h>
#include <string.h>

#include <vector>

#include "common.cuh"

namespace hcc {

static thread_local char g_err[512] = "";

void set_error(const char *fmt, ...) {
    va_list ap;
    va_start(ap, fmt);
    vsnprintf(g_err, sizeof g_err, fmt, ap);
    va_end(ap);
}

// ---------------------------------------------------------------------------------------
// conversion kernels
// ---------------------------------------------------------------------------------------

// Traversal records.  Nothing on the results depends on them: the hit a ray reports is defined
// by the triangle predicate alone (include/hcc.h), box culling only has to be conservative.
// The binary BVH is collapsed on the host into a 4-wide one (hcc_bvh_create: starting from a
// node's two children, the internal child with the largest surface area is replaced by its own
// two children until there are four or only leaves are left), so a ray makes about half as many
// dependent record fetches.  The k-th WIDE node owns one 64-byte record, two 256-bit loads:
//   w[3c .. 3c+2] = child c (0..3) x, y, z:  lo cell | hi cell << 16
//   w[12 + c]     = reference of child c
//   reference, internal child: (index of its wide node) + 1                       (bit 31 clear)
//   reference, leaf child    : 0x80000000 | (count-1) << 28 | first triangle slot, count <= 4 (a leaf of
//                              5..8 triangles gets a wide node of its own: two such halves, same box)
//   unused slot              : reference 0, box lo cell 32767 / hi cell 0 (never hit)
// Cells are indices of a uniform grid over the root box, g = (x - q_lo) * q_scale + 2 in fp32
// (a monotone map, so containment survives it), lo = floor(g) - 1, hi = ceil(g) + 1, clamped to
// [0, 32767]: every stored box contains the fp32 box with a margin of at least one cell
// (3e-5 of the scene extent), far above the rounding of the slab arithmetic in trace.cu.
__global__ void k_parents(const hcc_node *__restrict__ nodes, uint32_t n, uint32_t *__restrict__ parent) {
    uint32_t i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= n) return;
    hcc_node nd = nodes[i];
    if (nd.count == 0) {
        parent[nd.left_or_first] = i;
        parent[nd.left_or_first + 1u] = i;
    }
    if (i == 0) parent[0] = 0xFFFFFFFFu;
}

struct GridFrame { float lo[3], scale[3]; };

constexpr uint32_t WIDE_NONE = 0xFFFFFFFFu;

// wbox: per wide node and slot, the binary node whose box the slot carries (WIDE_NONE = unused slot);
// wref: the slot's reference, made on the host.
__global__ void k_build_wrec(const hcc_node *__restrict__ nodes, const uint32_t *__restrict__ wbox,
                             const uint32_t *__restrict__ wref, uint32_t n_wide, GridFrame f,
                             uint32_t *__restrict__ wrec) {
    uint32_t k = blockIdx.x * blockDim.x + threadIdx.x;
    if (k >= n_wide) return;
    uint32_t w[16];
    for (uint32_t c = 0; c < 4; ++c) {
        const uint32_t id = wbox[4 * (size_t)k + c];
        if (id == WIDE_NONE) {
            w[3 * c] = w[3 * c + 1] = w[3 * c + 2] = 0x00007FFFu;
            w[12 + c] = 0u;
            continue;
        }
        const hcc_node ch = nodes[id];
        for (int a = 0; a < 3; ++a) {
            const float gl = (ch.lo[a] - f.lo[a]) * f.scale[a] + HCC_GRID_OFFSET;
            const float gh = (ch.hi[a] - f.lo[a]) * f.scale[a] + HCC_GRID_OFFSET;
            // NaN or out-of-range boxes fall back to the whole axis (conservative)
            int ql = gl >= 1.0f ? (gl < 32768.0f ? (int)floorf(gl) - 1 : 32767) : 0;
            int qh = gh < 32766.0f ? (gh >= 0.0f ? (int)ceilf(gh) + 1 : 0) : 32767;
            if (!(gl == gl) || !(gh == gh)) { ql = 0; qh = 32767; }
            w[3 * c + a] = (uint32_t)ql | ((uint32_t)qh << 16);
        }
        w[12 + c] = wref[4 * (size_t)k + c];
    }
    uint4 *out = reinterpret_cast<uint4 *>(wrec + 16 * (size_t)k);
    for (int q = 0; q < 4; ++q) out[q] = make_uint4(w[4 * q], w[4 * q + 1], w[4 * q + 2], w[4 * q + 3]);
}

// Triangle record k (leaf order), 64 bytes so that it is two aligned 256-bit loads:
// (v0, prim id), (e1 = v1 - v0, 0), (e2 = v2 - v0, 0), padding.
__global__ void k_convert_tris(const float *__restrict__ tris, const uint32_t *__restrict__ prim_idx,
                               uint32_t n, float4 *__restrict__ out) {
    uint32_t k = blockIdx.x * blockDim.x + threadIdx.x;
    if (k >= n) return;
    uint32_t id = prim_idx[k];
    const float *v = tris + 9 * (size_t)id;
    float v0x = v[0], v0y = v[1], v0z = v[2];
    out[4 * (size_t)k + 0] = make_float4(v0x, v0y, v0z, __uint_as_float(id));
    out[4 * (size_t)k + 1] = make_float4(v[3] - v0x, v[4] - v0y, v[5] - v0z, 0.0f);
    out[4 * (size_t)k + 2] = make_float4(v[6] - v0x, v[7] - v0y, v[8] - v0z, 0.0f);
    out[4 * (size_t)k + 3] = make_float4(0.0f, 0.0f, 0.0f, 0.0f);
}

// Bottom-up pass: one thread per leaf walks to the root; at each parent the second
// thread to arrive continues (both children are final by then).  Computes the number
// of leaves below every node.
__global__ void k_subtree_leaves(const hcc_node *__restrict__ nodes, const uint32_t *__restrict__ parent,
                                 uint32_t *flags, uint32_t n, uint32_t *leaves) {
    uint32_t i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= n || nodes[i].count == 0) return;
    leaves[i] = 1u;
    uint32_t cur = i;
    while (cur != 0u) {
        uint32_t p = parent[cur];
        __threadfence();
        if (atomicAdd(&flags[p], 1u) == 0u) return;
        uint32_t l = nodes[p].left_or_first;
        leaves[p] = __ldcg(&leaves[l]) + __ldcg(&leaves[l + 1u]);
        cur = p;
    }
}

__device__ __forceinline__ float surface_area(const hcc_node &nd) {
    float dx = nd.hi[0] - nd.lo[0];
    float dy = nd.hi[1] - nd.lo[1];
    float dz = nd.hi[2] - nd.lo[2];
    return 2.0f * ((dx * dy + dy * dz) + dz * dx);
}

// Eq. 1, same bottom-up schedule.  Each node's value is computed exactly
// once from its two final children, so the result does not depend on thread timing.  The arrival
// mark of an internal node lives in its own slot of the OUTPUT array (zeroed by hcc_density first): the
// first child to arrive swaps 0 for HAD_PENDING and stops, the second finds the mark and writes the
// value, so concurrent calls on one BVH (different outputs, different streams) share no scratch.
constexpr uint32_t HAD_PENDING = 0xFFFFFFFFu;   // a NaN pattern no density takes
__global__ void k_density(const hcc_node *__restrict__ nodes, const uint32_t *__restrict__ parent,
                          uint32_t n, float lambda, float *had) {
    uint32_t i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= n) return;
    hcc_node nd = nodes[i];
    if (nd.count == 0) return;
    had[i] = (float)nd.count * surface_area(nd);
    uint32_t cur = i;
    while (cur != 0u) {
        uint32_t p = parent[cur];
        __threadfence();
        if (atomicCAS(reinterpret_cast<uint32_t *>(had) + p, 0u, HAD_PENDING) == 0u) return;
        hcc_node pn = nodes[p];
        float hl = __ldcg(&had[pn.left_or_first]);
        float hr = __ldcg(&had[pn.left_or_first + 1u]);
        __stcg(&had[p], (hl + hr) + (lambda * surface_area(pn)));
        cur = p;
    }
}

}  // namespace hcc

using namespace hcc;

extern "C" const char *hcc_last_error(void) { return hcc::g_err; }
extern "C" int32_t hcc_version(void) { return 100; }

extern "C" int32_t hcc_bvh_destroy(hcc_bvh *b) {
    if (!b) return HCC_OK;
    cudaFree(b->d_nodes);
    cudaFree(b->d_parent);
    cudaFree(b->d_leaves);
    cudaFree(b->d_flags);
    cudaFree(b->d_internal);
    cudaFree(b->d_wrec);
    cudaFree(b->d_trace_ctl);
    delete b->trace_calls;
    cudaFree(b->d_ttri);
    delete b;
    return HCC_OK;
}

extern "C" int32_t hcc_bvh_create(const hcc_node *nodes, uint32_t n_nodes, const float *tris, uint32_t n_tris,
                                  const uint32_t *prim_idx, void *stream, hcc_bvh **out) {
    HCC_REQUIRE(nodes && tris && prim_idx && out, HCC_ERR_INVALID_ARG, "hcc_bvh_create: NULL argument");
    HCC_REQUIRE(n_nodes >= 1 && n_tris >= 1, HCC_ERR_INVALID_ARG, "hcc_bvh_create: empty BVH");
    HCC_REQUIRE(n_tris < (1u << 27) && n_nodes < (1u << 30), HCC_ERR_UNSUPPORTED,
                "hcc_bvh_create: more than 2^27 triangles or 2^30 nodes");
    *out = nullptr;
    cudaStream_t s = (cudaStream_t)stream;

    // ---- host validation: one pass in index order (parent < child makes depth a prefix computation)
    std::vector<uint32_t> depth(n_nodes, 0u);
    std::vector<uint8_t> seen(n_nodes, 0), tri_seen(n_tris, 0);
    std::vector<uint32_t> internal_ids;
    internal_ids.reserve(n_nodes / 2 + 1);
    uint32_t max_depth = 0, n_leaves = 0;
    uint64_t tri_total = 0;
    seen[0] = 1;
    for (uint32_t i = 0; i < n_nodes; ++i) {
        const hcc_node &nd = nodes[i];
        HCC_REQUIRE(seen[i], HCC_ERR_INVALID_ARG, "hcc_bvh_create: node %u is not reachable from the root", i);
        if (depth[i] > max_depth) max_depth = depth[i];
        if (nd.count == 0) {
            uint32_t l = nd.left_or_first;
            internal_ids.push_back(i);
            HCC_REQUIRE(l > i && (uint64_t)l + 1u < n_nodes, HCC_ERR_INVALID_ARG,
                        "hcc_bvh_create: node %u has children out of range or not after it", i);
            HCC_REQUIRE(!seen[l] && !seen[l + 1], HCC_ERR_INVALID_ARG, "hcc_bvh_create: node %u shares a child", i);
            seen[l] = seen[l + 1] = 1;
            depth[l] = depth[l + 1] = depth[i] + 1u;
        } else {
            ++n_leaves;
            HCC_REQUIRE(nd.count <= 8u, HCC_ERR_UNSUPPORTED, "hcc_bvh_create: leaf %u holds %u > 8 triangles", i, nd.count);
            HCC_REQUIRE((uint64_t)nd.left_or_first + nd.count <= n_tris, HCC_ERR_INVALID_ARG,
                        "hcc_bvh_create: leaf %u triangle range out of bounds", i);
            tri_total += nd.count;
        }
    }
    for (uint32_t k = 0; k < n_tris; ++k) {
        HCC_REQUIRE(prim_idx[k] < n_tris, HCC_ERR_INVALID_ARG, "hcc_bvh_create: prim_idx[%u] out of range", k);
        tri_seen[prim_idx[k]] = 1;
    }
    HCC_REQUIRE(max_depth <= 63u, HCC_ERR_UNSUPPORTED, "hcc_bvh_create: BVH depth %u > 63", max_depth);
    (void)tri_total;

    hcc_bvh *b = new hcc_bvh();
    memset(b, 0, sizeof *b);
    b->n_nodes = n_nodes; b->n_tris = n_tris; b->n_leaves = n_leaves; b->max_depth = max_depth;
    for (int a = 0; a < 3; ++a) { b->scene_lo[a] = nodes[0].lo[a]; b->scene_hi[a] = nodes[0].hi[a]; }

    // traversal grid over the root box and the root's traversal reference
    GridFrame frame;
    for (int a = 0; a < 3; ++a) {
        const float ext = b->scene_hi[a] - b->scene_lo[a];
        b->q_lo[a] = frame.lo[a] = b->scene_lo[a];
        b->q_scale[a] = frame.scale[a] = ext > 0.0f && HCC_GRID_CELLS / ext < 3.0e38f ? HCC_GRID_CELLS / ext : 0.0f;
    }
    b->n_internal = (uint32_t)internal_ids.size();
    b->trace_calls = new std::atomic<uint32_t>(0u);

    // ---- collapse to a 4-wide tree (host, one pass): wide node ids are handed out family by family
    //      (the internal children of one wide node are neighbours) in depth-first order
    std::vector<uint32_t> wbox, wref;
    {
        auto area = [&](uint32_t i) {
            const hcc_node &nd = nodes[i];
            const float dx = nd.hi[0] - nd.lo[0], dy = nd.hi[1] - nd.lo[1], dz = nd.hi[2] - nd.lo[2];
            return dx * dy + dy * dz + dz * dx;
        };
        auto leaf_ref = [](uint32_t first, uint32_t count) { return HCC_REF_LEAF | ((count - 1u) << 28) | first; };
        uint32_t n_wide = 0;
        auto new_wide = [&]() {
            wbox.resize(4 * (size_t)(n_wide + 1), WIDE_NONE);
            wref.resize(4 * (size_t)(n_wide + 1), 0u);
            return n_wide++;
        };
        // reference of binary node i as a child (or as the root); internal nodes are queued for expansion
        std::vector<std::pair<uint32_t, uint32_t>> todo;        // (wide node, binary node heading it)
        auto ref_of = [&](uint32_t i) -> uint32_t {
            const hcc_node &nd = nodes[i];
            if (nd.count == 0) return new_wide() + 1u;
            if (nd.count <= 4u) return leaf_ref(nd.left_or_first, nd.count);
            const uint32_t w = new_wide();          // a big leaf: two halves under its own box
            wbox[4 * (size_t)w] = wbox[4 * (size_t)w + 1] = i;
            wref[4 * (size_t)w] = leaf_ref(nd.left_or_first, 4u);
            wref[4 * (size_t)w + 1] = leaf_ref(nd.left_or_first + 4u, nd.count - 4u);
            return w + 1u;
        };
        wbox.reserve(4 * (size_t)(n_nodes / 3 + 2));
        wref.reserve(4 * (size_t)(n_nodes / 3 + 2));
        // the root reference is always a wide node (trace.cu never holds a leaf reference as its current
        // node): a root leaf of up to four triangles becomes the only child of a wide node of its own
        if (nodes[0].count != 0 && nodes[0].count <= 4u) {
            const uint32_t w = new_wide();
            wbox[4 * (size_t)w] = 0u;
            wref[4 * (size_t)w] = leaf_ref(nodes[0].left_or_first, nodes[0].count);
            b->root_ref = w + 1u;
        } else {
            b->root_ref = ref_of(0u);
        }
        if (nodes[0].count == 0) todo.push_back({b->root_ref - 1u, 0u});
        while (!todo.empty()) {
            const uint32_t wide = todo.back().first, head = todo.back().second;
            todo.pop_back();
            uint32_t c[4] = {nodes[head].left_or_first, nodes[head].left_or_first + 1u, WIDE_NONE, WIDE_NONE};
            uint32_t nc = 2;
            while (nc < 4) {
                int pick = -1;
                float best = -1.0f;
                for (uint32_t k = 0; k < nc; ++k)
                    if (nodes[c[k]].count == 0) {
                        const float a = area(c[k]);
                        if (pick < 0 || a > best) { pick = (int)k; best = a; }
                    }
                if (pick < 0) break;
                const uint32_t l = nodes[c[pick]].left_or_first;
                c[pick] = l;
                c[nc++] = l + 1u;
            }
            uint32_t refs[4];
            for (uint32_t k = 0; k < nc; ++k) refs[k] = ref_of(c[k]);    // may grow wbox / wref
            for (uint32_t k = 0; k < nc; ++k) {
                wbox[4 * (size_t)wide + k] = c[k];
                wref[4 * (size_t)wide + k] = refs[k];
            }
            for (uint32_t k = nc; k-- > 0;)
                if (nodes[c[k]].count == 0) todo.push_back({refs[k] - 1u, c[k]});
        }
        b->n_wide = n_wide;
    }

    float *d_tris = nullptr;
    uint32_t *d_prim = nullptr, *d_wbox = nullptr, *d_wref = nullptr;
    cudaError_t e = cudaSuccess;
    auto alloc = [&](void **p, size_t bytes) { if (e == cudaSuccess) e = cudaMalloc(p, bytes); };
    alloc((void **)&b->d_nodes, sizeof(hcc_node) * (size_t)n_nodes);
    alloc((void **)&b->d_parent, sizeof(uint32_t) * (size_t)n_nodes);
    alloc((void **)&b->d_leaves, sizeof(uint32_t) * (size_t)n_nodes);
    alloc((void **)&b->d_flags, sizeof(uint32_t) * (size_t)n_nodes);
    alloc((void **)&b->d_internal, sizeof(uint32_t) * (internal_ids.size() + 1));
    alloc((void **)&b->d_wrec, 64 * ((size_t)b->n_wide + 1));
    alloc((void **)&b->d_trace_ctl, 2 * HCC_TRACE_SLOTS * sizeof(uint32_t));
    alloc((void **)&b->d_ttri, sizeof(float4) * 4 * (size_t)n_tris);
    alloc((void **)&d_wbox, sizeof(uint32_t) * (wbox.size() + 4));
    alloc((void **)&d_wref, sizeof(uint32_t) * (wref.size() + 4));
    alloc((void **)&d_tris, sizeof(float) * 9 * (size_t)n_tris);
    alloc((void **)&d_prim, sizeof(uint32_t) * (size_t)n_tris);
    if (e != cudaSuccess) {
        set_error("hcc_bvh_create: cudaMalloc failed: %s", cudaGetErrorString(e));
        cudaFree(d_tris); cudaFree(d_prim); cudaFree(d_wbox); cudaFree(d_wref);
        hcc_bvh_destroy(b);
        return e == cudaErrorMemoryAllocation ? HCC_ERR_OUT_OF_MEMORY : HCC_ERR_CUDA;
    }
    auto fail = [&](cudaError_t err, const char *what) {
        set_error("hcc_bvh_create: %s: %s", what, cudaGetErrorString(err));
        cudaFree(d_tris); cudaFree(d_prim); cudaFree(d_wbox); cudaFree(d_wref);
        hcc_bvh_destroy(b);
        return (int32_t)HCC_ERR_CUDA;
    };
    if ((e = cudaMemcpyAsync(b->d_nodes, nodes, sizeof(hcc_node) * (size_t)n_nodes, cudaMemcpyHostToDevice, s)) != cudaSuccess) return fail(e, "copy nodes");
    if ((e = cudaMemcpyAsync(d_tris, tris, sizeof(float) * 9 * (size_t)n_tris, cudaMemcpyHostToDevice, s)) != cudaSuccess) return fail(e, "copy triangles");
    if ((e = cudaMemcpyAsync(d_prim, prim_idx, sizeof(uint32_t) * (size_t)n_tris, cudaMemcpyHostToDevice, s)) != cudaSuccess) return fail(e, "copy prim_idx");
    if (!wbox.empty() &&
        ((e = cudaMemcpyAsync(d_wbox, wbox.data(), sizeof(uint32_t) * wbox.size(), cudaMemcpyHostToDevice, s)) != cudaSuccess ||
         (e = cudaMemcpyAsync(d_wref, wref.data(), sizeof(uint32_t) * wref.size(), cudaMemcpyHostToDevice, s)) != cudaSuccess))
        return fail(e, "copy wide nodes");
    if (!internal_ids.empty() &&
        (e = cudaMemcpyAsync(b->d_internal, internal_ids.data(), sizeof(uint32_t) * internal_ids.size(), cudaMemcpyHostToDevice, s)) != cudaSuccess) return fail(e, "copy internal ids");
    if ((e = cudaMemsetAsync(b->d_flags, 0, sizeof(uint32_t) * (size_t)n_nodes, s)) != cudaSuccess) return fail(e, "memset");
    if ((e = cudaMemsetAsync(b->d_trace_ctl, 0, 2 * HCC_TRACE_SLOTS * sizeof(uint32_t), s)) != cudaSuccess) return fail(e, "memset");
    const uint32_t T = 256;
    k_parents<<<(n_nodes + T - 1) / T, T, 0, s>>>(b->d_nodes, n_nodes, b->d_parent);
    if (b->n_wide)
        k_build_wrec<<<(b->n_wide + T - 1) / T, T, 0, s>>>(b->d_nodes, d_wbox, d_wref, b->n_wide, frame, b->d_wrec);
    k_convert_tris<<<(n_tris + T - 1) / T, T, 0, s>>>(d_tris, d_prim, n_tris, b->d_ttri);
    k_subtree_leaves<<<(n_nodes + T - 1) / T, T, 0, s>>>(b->d_nodes, b->d_parent, b->d_flags, n_nodes, b->d_leaves);
    if ((e = cudaGetLastError()) != cudaSuccess) return fail(e, "conversion kernels");
    if ((e = cudaStreamSynchronize(s)) != cudaSuccess) return fail(e, "synchronise");
    cudaFree(d_tris);
    cudaFree(d_prim);
    cudaFree(d_wbox);
    cudaFree(d_wref);
    *out = b;
    return HCC_OK;
}

extern "C" int32_t hcc_bvh_info(const hcc_bvh *b, uint32_t *n_nodes, uint32_t *n_tris, uint32_t *n_leaves,
                                uint32_t *max_depth, float scene_lo[3], float scene_hi[3]) {
    HCC_REQUIRE(b, HCC_ERR_INVALID_ARG, "hcc_bvh_info: NULL bvh");
    if (n_nodes) *n_nodes = b->n_nodes;
    if (n_tris) *n_tris = b->n_tris;
    if (n_leaves) *n_leaves = b->n_leaves;
    if (max_depth) *max_depth = b->max_depth;
    for (int a = 0; a < 3; ++a) {
        if (scene_lo) scene_lo[a] = b->scene_lo[a];
        if (scene_hi) scene_hi[a] = b->scene_hi[a];
    }
    return HCC_OK;
}

extern "C" int32_t hcc_density(const hcc_bvh *b, float lambda, float *density_dev, void *stream) {
    HCC_REQUIRE(b && density_dev, HCC_ERR_INVALID_ARG, "hcc_density: NULL argument");
    HCC_REQUIRE(aligned(density_dev, 16), HCC_ERR_BAD_ALIGNMENT, "hcc_density: density_dev not 16-byte aligned");
    HCC_REQUIRE(lambda >= 0.0f, HCC_ERR_INVALID_ARG, "hcc_density: lambda must be >= 0");
    cudaStream_t s = (cudaStream_t)stream;
    HCC_CUDA_TRY(cudaMemsetAsync(density_dev, 0, sizeof(float) * (size_t)b->n_nodes, s));
    const uint32_t T = 256;
    k_density<<<(b->n_nodes + T - 1) / T, T, 0, s>>>(b->d_nodes, b->d_parent, b->n_nodes, lambda, density_dev);
    HCC_CUDA_TRY(cudaGetLastError());
    return HCC_OK;
}
