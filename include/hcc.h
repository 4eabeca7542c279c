/* hcc.h — C ABI of the B200-native hierarchy-cut-code ray-reordering hot path.
 *
 * Paper: "Faster Ray Tracing through Hierarchy Cut Code", arxiv 2305.16652
 * (cited as PAPER.md:<line>).  The path (Figure 11; pre-process
 * :155-192):  density + cut selection -> key computation -> sort of ray indices ->
 * trace through the sorted indices.  Every step runs in CUDA kernels written for
 * sm_100a; there is no CPU fallback.
 *
 * Conventions
 *  - Every function returns an int32 status: HCC_OK (0) or a negative hcc_status.
 *    Nothing throws or aborts across this boundary; hcc_last_error() returns the
 *    calling thread's last message.
 *  - `stream` is a cudaStream_t passed as void* (NULL = the legacy default stream).
 *    Calls that take a stream only ENQUEUE work on it and return; they never
 *    allocate or free device memory.  Allocation happens in *_create only.
 *  - "dev" pointers are device pointers owned by the caller (e.g. torch tensors);
 *    "host" pointers are host memory read during the call.  Handles (hcc_bvh,
 *    hcc_cut) are owned by the library and released with *_destroy.
 *  - Alignment: rays 32 bytes; keys, perm, hits, density, workspace 16 bytes.
 *    A misaligned pointer returns HCC_ERR_BAD_ALIGNMENT.
 *  - n = 0 is valid everywhere and is a no-op.
 *
 * Layouts
 *  - node (canonical BVH, 32 bytes): { float lo[3], hi[3]; uint32 left_or_first;
 *    uint32 count }.  count == 0: internal, children are nodes left_or_first and
 *    left_or_first + 1 (siblings adjacent, parent index < child index, root = 0).
 *    count > 0: leaf holding triangles prim_idx[left_or_first .. +count), count <= 8.
 *  - triangle: 9 floats v0 v1 v2; prim ids index this array.
 *  - ray (32 bytes, AoS): { ox, oy, oz, tmin, dx, dy, dz, tmax }.  d should be unit
 *    length for TwoPoint (PAPER.md:241 fixed-length estimate); traversal and HCC do
 *    not require it.
 *  - key: uint32 when the cut's / call's key_bits <= 32, else uint64; right-aligned
 *    (all bits above bits_used are zero).
 *  - closest hit (16 bytes): { float t; uint32 prim; float u; float v }, t = +inf and
 *    prim = 0xFFFFFFFF on a miss.   any hit: one uint8 per ray (1 = occluded).
 */
#ifndef HCC_H
#define HCC_H

#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

/* Exported symbols (the library is built with -fvisibility=hidden). */
#if defined(__GNUC__)
#define HCC_API __attribute__((visibility("default")))
#else
#define HCC_API
#endif

#define HCC_MAX_LEVELS 16u
#define HCC_MAX_WIDTH 64u
#define HCC_MISS_PRIM 0xFFFFFFFFu

typedef enum hcc_status {
    HCC_OK = 0,
    HCC_ERR_INVALID_ARG = -1,
    HCC_ERR_BAD_ALIGNMENT = -2,
    HCC_ERR_OUT_OF_MEMORY = -3,
    HCC_ERR_CUDA = -4,
    HCC_ERR_UNSUPPORTED = -5
} hcc_status;

typedef enum hcc_trace_mode { HCC_TRACE_CLOSEST = 0, HCC_TRACE_ANY = 1 } hcc_trace_mode;

/* The three ray orders compared throughout the paper's Tables 2-3. */
typedef enum hcc_order { HCC_ORDER_NOSORT = 0, HCC_ORDER_TWOPOINT = 1, HCC_ORDER_HCC = 2 } hcc_order;

typedef struct hcc_node {
    float lo[3];
    float hi[3];
    uint32_t left_or_first;
    uint32_t count;
} hcc_node;

typedef struct hcc_hit {
    float t;
    uint32_t prim;
    float u;
    float v;
} hcc_hit;

typedef struct hcc_bvh hcc_bvh; /* opaque: device copy of the BVH in the GPU layouts */
typedef struct hcc_cut hcc_cut; /* opaque: device level tables of one cut hierarchy  */
typedef struct hcc_pipeline hcc_pipeline; /* opaque: per-batch scratch (keys, perm, sort workspace) */

/* Message of the last error on the calling thread ("" if none). Never NULL. */
HCC_API const char *hcc_last_error(void);

/* Library version (major*10000 + minor*100 + patch). */
HCC_API int32_t hcc_version(void);

/* ---- BVH ---------------------------------------------------------------------------
 * The BVH is INPUT (BASELINE.json north_star: built by a deterministic host binned-SAH
 * builder); the paper assumes a SAH BVH and does not describe a builder.
 * hcc_bvh_create validates the canonical arrays on the host (indices in range, siblings
 * adjacent, parent < child, every node reachable once, leaf count in 1..8, depth <= 63,
 * fewer than 2^27 triangles and 2^30 nodes:
 * otherwise HCC_ERR_INVALID_ARG / HCC_ERR_UNSUPPORTED), copies them to the device and runs
 * the conversion kernels on `stream`: the binary tree is collapsed on the host into a 4-wide
 * traversal tree (the internal child with the largest surface area is opened until a node has
 * four children) with one 64-byte record per wide node (four child boxes as 15-bit cells of a
 * uniform grid over the root box, rounded outwards and padded by one cell, plus the four child
 * references; a leaf of 5..8 triangles becomes two leaves under a wide node of its own), the
 * 64-byte triangle records in leaf order, parent links and sub-tree leaf counts.  The quantised boxes only cull: results
 * are defined by the triangle predicate under hcc_trace.  All three arrays are host pointers, read before return.
 * The call synchronises `stream` before returning. */
HCC_API int32_t hcc_bvh_create(const hcc_node *nodes_host, uint32_t n_nodes, const float *tris_host,
                       uint32_t n_tris, const uint32_t *prim_idx_host, void *stream,
                       hcc_bvh **out);
HCC_API int32_t hcc_bvh_destroy(hcc_bvh *bvh);
/* Any out pointer may be NULL.  scene_lo/hi = the root box. */
HCC_API int32_t hcc_bvh_info(const hcc_bvh *bvh, uint32_t *n_nodes, uint32_t *n_tris, uint32_t *n_leaves,
                     uint32_t *max_depth, float scene_lo[3], float scene_hi[3]);

/* ---- (a1) density + cut selection ------------------------------------------------------
 * hcc_density: hierarchically accumulated density, Eq. 1 (:187):
 *   leaf  HAD = TC * SA;  internal  HAD = (HAD_left + HAD_right) + lambda * SA,
 *   SA = 2((dx*dy + dy*dz) + dz*dx), every operation one rounded fp32 operation.
 * density_dev: float32[n_nodes], written (also used as the pass's own scratch, so calls on one BVH with
 * different outputs may run concurrently).  The paper uses lambda = 0.125 (:185, :276). */
HCC_API int32_t hcc_density(const hcc_bvh *bvh, float lambda, float *density_dev, void *stream);

/* A cut handle with room for hierarchies of up to max_K finest-level nodes. */
HCC_API int32_t hcc_cut_create(uint32_t max_K, hcc_cut **out);
HCC_API int32_t hcc_cut_destroy(hcc_cut *cut);

/* hcc_select_cut: the K-node cut of the BVH by priority-queue search on `density_dev`
 * (Algorithm 2; cut nodes ordered by density descending, :192), stored
 * as the level tables the encoder reads.  K <= key_bits gives one level = plain HCC
 * (:146-153, :206).  K > key_bits gives the multi-level compressed code (:204-237): the
 * fewest levels m >= 2 of power-of-two widths, the exponent of K split as evenly as
 * possible (larger first), with sum(widths) <= key_bits; K = (key_bits/2)^2 is the paper's
 * two-level MLHCC (:216, :220).  If no split fits, K is halved until one does; the K
 * actually used is reported by hcc_cut_info.  Each table is built by Algorithm 3 (:222-231)
 * started at its parent entry, with "large enough sub-tree" = at least as many leaves as the
 * next level's width; a node that is not large enough is kept as an entry (not dropped).
 * Ties in density break toward the lower node index.
 * key_bits must be one of 16, 24, 32, 48, 64; K >= 1; else HCC_ERR_INVALID_ARG.
 * density_dev: float32[n_nodes] (read).  Results stay on the device. */
HCC_API int32_t hcc_select_cut(const hcc_bvh *bvh, const float *density_dev, uint32_t K, uint32_t key_bits,
                       hcc_cut *cut, void *stream);
/* Same with explicit level widths (each 1..64, m <= HCC_MAX_LEVELS, sum <= key_bits). */
HCC_API int32_t hcc_select_cut_levels(const hcc_bvh *bvh, const float *density_dev, const uint32_t *widths_host,
                              uint32_t m, uint32_t key_bits, hcc_cut *cut, void *stream);

/* (f4) The same with flags.  HCC_CUT_ALG3_DISCARD: every level that has a level below it is built by
 * Algorithm 3 as printed ("we discard the top-level node that does not have a
 * sufficient subtree ... This ensures that there are no empty low-level nodes"): a popped node with fewer
 * leaves below it than the next level's width is dropped instead of being kept as an entry.  Tables may
 * then hold fewer entries, leave parts of the scene covered by no entry, or be empty; the last level is
 * Algorithm 2 either way.  flags = 0 is hcc_select_cut_levels. */
#define HCC_CUT_ALG3_DISCARD 1u
HCC_API int32_t hcc_select_cut_levels_ex(const hcc_bvh *bvh, const float *density_dev, const uint32_t *widths,
                                 uint32_t m, uint32_t key_bits, uint32_t flags, hcc_cut *cut, void *stream);
/* Shape of the last selection (host values, no synchronisation): number of levels, their
 * widths (array of HCC_MAX_LEVELS), K actually used, key bits used = sum of widths, key
 * container bits (32 or 64), total entries and tables over all levels. Out pointers may be NULL. */
HCC_API int32_t hcc_cut_info(const hcc_cut *cut, uint32_t *m, uint32_t *widths, uint32_t *K_eff,
                     uint32_t *bits_used, uint32_t *container_bits, uint64_t *n_entries,
                     uint64_t *n_tables);
/* Copy the tables to the host for inspection: entry_node_host[n_entries] (node ids, levels
 * concatenated, table t of level l at offset ent_off[l] + t*w[l], 0xFFFFFFFF = empty slot)
 * and table_cnt_host[n_tables].  Synchronises `stream`. */
HCC_API int32_t hcc_cut_read(const hcc_cut *cut, uint32_t *entry_node_host, uint32_t *table_cnt_host,
                     void *stream);

/* Algorithm 2 verbatim for ANY K, as its data-parallel closed form:
 * because the density of a parent is >= that of its children and popping a leaf never
 * advances the loop, the cut is the set of children of the K-1 highest-density internal
 * nodes that are not themselves among those K-1 (ties -> lower index).  Implemented as a
 * radix sort of the internal nodes by density plus a flag/compact pass and a final sort by
 * density (:192).  cut_nodes_dev: uint32[K] written with the node ids, density descending;
 * count_dev: uint32[1] = number written = min(K, #leaves).  workspace from
 * hcc_select_cut_flat_workspace_bytes. */
HCC_API int32_t hcc_select_cut_flat_workspace_bytes(const hcc_bvh *bvh, uint32_t K, uint64_t *bytes);
HCC_API int32_t hcc_select_cut_flat(const hcc_bvh *bvh, const float *density_dev, uint32_t K,
                            uint32_t *cut_nodes_dev, uint32_t *count_dev, void *workspace_dev,
                            uint64_t workspace_bytes, void *stream);

/* ---- (a2) encode ----------------------------------------------------------------------
 * hcc_encode: the hierarchy cut code of every ray (Algorithm 1; levels
 * below the first :208, :218-220).  Bit for entry j of a level = [ray hits that node's
 * box], entry 0 (highest density) in the field's most significant bit (:192, :202); the top
 * level's field is the most significant, each further level directly below (:216, :220);
 * the representative of a level is its first hit entry (:218); a level with no hit zeroes
 * all lower fields.  Box test: inv = 1/d; t1 = (lo-o)*inv, t2 = (hi-o)*inv per axis,
 * tn = max(tmin, max_a min(t1,t2)), tf = min(tmax, min_a max(t1,t2)), hit <=> tn <= tf,
 * IEEE fp32 operation by operation with NaN-dropping min/max.
 * keys_dev: uint32[n] if the cut's container is 32 bits, else uint64[n]. */
HCC_API int32_t hcc_encode(const float *rays_dev, uint64_t n, const hcc_cut *cut, void *keys_dev, void *stream);

/* TwoPoint comparison path: origin and estimated end point
 * o + (0.25 * largest scene extent) * d, each coordinate quantised to floor(key_bits/6)
 * bits inside [scene_lo, scene_hi] and bit-interleaved o.x o.y o.z t.x t.y t.z from the
 * most significant bit down.  keys_dev: uint32[n] if key_bits <= 32 else uint64[n]. */
HCC_API int32_t hcc_encode_twopoint(const float *rays_dev, uint64_t n, const float scene_lo[3],
                            const float scene_hi[3], uint32_t key_bits, void *keys_dev, void *stream);

/* ---- NEXT rows of the scope table -------------------------------------------
 * (f3) Prefix path code, PAPER.md:116-128 (section 4.1, Figure 5): "setting each bit to 1 if the
 * corresponding node intersection result is true, and 0 otherwise ... when the rays are forced
 * to traverse the BVH in the same order", the walk ended after key_bits tests.  The walk: depth
 * first, left child before right, starting with the root's own test; every node visited gets the
 * slab test of hcc_encode on the ray's [tmin, tmax] and contributes one bit, the first test in
 * bit key_bits-1; a hit internal node has its children visited next, a hit leaf nothing more (no
 * triangle tests); an exhausted walk leaves the remaining low bits zero.  The paper's upper-bound
 * ordering, not a practical one (:128).  keys_dev: uint32[n] if key_bits <= 32 else uint64[n]. */
HCC_API int32_t hcc_encode_ppc(const hcc_bvh *bvh, const float *rays_dev, uint64_t n, uint32_t key_bits,
                       void *keys_dev, void *stream);

/* (f4) Regular grid encoding: "the BVH cut nodes are replaced by grids that divide
 * the space evenly".  Fills `cut` with level tables of the given widths (powers of two >= 2, sum
 * <= key_bits) whose entries are cells of a regular subdivision of the root box, so hcc_encode
 * and the rest of the path run unchanged.  A cell is named by its path of halvings; halving i
 * (counted from the root, across levels) splits axis i mod 3, bit 0 = lower half; entry j of a
 * table is the cell whose path bits of that level are j (first halving in the top bit).  With
 * n_a halvings of axis a and cell index i_a:  lo_a = scene_lo_a + (scene_hi_a - scene_lo_a) *
 * (i_a / 2^n_a) (fp32, three operations), hi_a likewise at i_a + 1, exactly scene_hi_a for the
 * last cell.  All tables are full; hcc_cut_read returns HCC_INVALID_NODE for every entry. */
HCC_API int32_t hcc_select_grid(const hcc_bvh *bvh, const uint32_t *widths, uint32_t m, uint32_t key_bits,
                        hcc_cut *cut, void *stream);

/* Boxes of all table entries of `cut` as 6 floats (lo.xyz, hi.xyz) each, in entry order (host). */
HCC_API int32_t hcc_cut_read_boxes(const hcc_cut *cut, float *boxes_host, void *stream);

/* ---- (a3) sort ------------------------------------------------------------------------
 * Stable ascending order of ray ids by key ("sorting the HCCs as natural
 * numbers", :247 "sorts the indices of rays"): perm_dev[j] = id of the ray at rank j; equal
 * keys keep ascending id.  LSD radix sort, 8-bit digits, one chained-scan ("onesweep") pass
 * per digit over bits [0, bits_used); bits above bits_used must be zero.
 * keys_dev (container_bits = 32 or 64) is clobbered.  n < 2^30.
 * workspace_dev: at least hcc_sort_workspace_bytes(n, container_bits) bytes. */
HCC_API int32_t hcc_sort_workspace_bytes(uint64_t n, uint32_t container_bits, uint64_t *bytes);
HCC_API int32_t hcc_sort(void *keys_dev, uint64_t n, uint32_t container_bits, uint32_t bits_used,
                 uint32_t *perm_dev, void *workspace_dev, uint64_t workspace_bytes, void *stream);

/* Sort-cost reduction the paper proposes (§6.6.1 "skip the last few bits during
 * encoding and terminate bucket sorting early"): the stable ascending order by the key bits
 * [bit_lo, bit_hi) only, i.e. by (key >> bit_lo); bits at and above bit_hi must be zero.  Rays
 * whose keys differ only below bit_lo keep their input order.  ceil((bit_hi - bit_lo) / 8) radix
 * passes.  hcc_sort(.., bits_used, ..) == hcc_sort_range(.., 0, bits_used, ..).  Other arguments,
 * workspace and errors as hcc_sort. */
HCC_API int32_t hcc_sort_range(void *keys_dev, uint64_t n, uint32_t container_bits, uint32_t bit_lo, uint32_t bit_hi,
                       uint32_t *perm_dev, void *workspace_dev, uint64_t workspace_bytes, void *stream);

/* hcc_sort for callers that have no way to obtain device memory for a workspace.  Some users of this
 * library sit where cudaMalloc is off limits: a plug-in running under a host application that owns the
 * GPU's memory pool and hands the plug-in only its input and output buffers, a real-time render loop that
 * must not take the driver's allocation lock, a worker started after its parent has already committed all
 * of HBM.  For them the sort's workspace (the second key / ray-id buffers of the ping-pong, the digit
 * histograms and the look-back status rows) lives in a fixed array that is part of
 * the library image itself: every GPU on which the library's kernels are loaded carries
 * HCC_SORT_STATIC_BYTES (4 MiB) for it until the process exits, whether or not this call is ever used.
 * That is why the limit is small: n <= HCC_SORT_STATIC_MAX_N (262,144 pairs, either key width); a larger
 * n returns HCC_ERR_UNSUPPORTED with a message naming the limit, and nothing is enqueued.
 *
 * Same result as hcc_sort(keys_dev, n, container_bits, bits_used, perm_dev, <workspace>, .., stream),
 * bit for bit; keys_dev is clobbered; the caller still owns keys_dev and perm_dev.  The call makes no
 * cudaMalloc / cudaFree and calls nothing that does.
 *  - First call on a device: with that device current, the call looks up the array's device address and
 *    sets the sort kernels' shared-memory attribute (both cached per device).  Make that first call outside
 *    any stream capture.
 *  - There is ONE array per device, shared by every call from every thread.  Two hcc_sort_static calls
 *    whose kernels can overlap on the GPU (different streams without an ordering between them) race on it
 *    and give garbage; calls on one stream, or ordered by events, are fine.  The array keeps whatever the
 *    previous call left in it; the first kernel of each call clears the part that has to start at zero
 *    (histograms, tickets, status rows), so no call depends on an earlier one. */
#define HCC_SORT_STATIC_MAX_N 262144u
#define HCC_SORT_STATIC_BYTES 4194304u
HCC_API int32_t hcc_sort_static(void *keys_dev, uint64_t n, uint32_t container_bits, uint32_t bits_used,
                        uint32_t *perm_dev, void *stream);

/* ---- (a4) trace -----------------------------------------------------------------------
 * Rays are traced through perm_dev (perm_dev == NULL: the input order 0, 1, ..., the NoSort
 * order): warps take 32-rank chunks of consecutive ranks, so the rays a warp holds are
 * neighbours in the given order, and every result is written at the ray's own index
 * ("the trace kernel fetches the rays based on these sorted indices").  The chunks
 * of a permutation are handed out from its END (descending keys: hierarchy cut codes carry the
 * densest cut nodes in their top bits, so the rays with the most traversal work start first and
 * the kernel runs out on cheap ones); which warp traces which chunk when has no effect on any
 * result.  n < 2^32 - 2^24.  Up to 1024 trace launches on one hcc_bvh may be in flight at a
 * time (each takes its own work counter, zeroed on `stream` by a kernel of the call).  The quantised
 * boxes are tested with a slack proportional to the distance of the ray origin from the scene
 * (2^-20 of it), which covers the fp32 rounding of the plane distances for origins up to about
 * 10^4 scene extents away; beyond that a triangle may be culled that the predicate would accept.  CLOSEST: hits_dev = hcc_hit[n]: the triangle with the
 * smallest t in (tmin, tmax), ties to the lowest prim id.  ANY: hits_dev = uint8[n].
 * Triangle test (fp32, fmaf where written): e1 = v1-v0, e2 = v2-v0, p = d x e2,
 * det = e1.p (0 -> miss), inv = 1/det, s = o-v0, u = (s.p)*inv, q = s x e1, v = (d.q)*inv,
 * t = (e2.q)*inv; hit <=> u >= 0, v >= 0, u+v <= 1, tmin < t < tmax; with
 * cross(a,b).x = fmaf(a.y,b.z,-(a.z*b.y)) and dot(a,b) = fmaf(a.x,b.x,fmaf(a.y,b.y,a.z*b.z)). */
HCC_API int32_t hcc_trace(const hcc_bvh *bvh, const float *rays_dev, uint64_t n, const uint32_t *perm_dev,
                  int32_t mode, void *hits_dev, void *stream);

/* Same traversal, instrumented (never used for timing): stats_dev = uint64[8], zeroed by the
 * call, then [0] = wide-node records fetched by rays (64 bytes each), [1] = triangle records
 * fetched (64 bytes each), [2] = rays traced, [3] = deepest traversal stack, and per WARP-level
 * node step (the 32 rays a warp holds fetch their records with one load instruction): [4] =
 * distinct records fetched, summed over steps, [5] = steps, [6] = lanes taking part, summed.
 * [4]/[5] is what a coherent order lowers (rays of a warp sharing node
 * fetches); [0] hardly depends on the order.  [7] = warp-level triangle rounds ([1]/[7] =
 * triangle tests per round).  hits_dev as hcc_trace. */
HCC_API int32_t hcc_trace_stats(const hcc_bvh *bvh, const float *rays_dev, uint64_t n, const uint32_t *perm_dev,
                        int32_t mode, void *hits_dev, uint64_t *stats_dev, void *stream);

/* ---- the per-batch path as one call -----------------------------------------------------
 * PAPER.md:245-247 (Figure 11): key compute kernel -> ray sort kernel -> trace kernel, per
 * ray batch.  A pipeline handle owns the scratch for batches of up to n_max rays (keys, perm,
 * the sort workspace; with HCC_PIPELINE_HOST_STAGING a device copy of the rays and hits for the
 * host-buffer calls; with HCC_PIPELINE_PAIR a second key buffer and sort workspace, a stream
 * and two events for hcc_reorder_trace_pair), so a call allocates nothing.
 * container_bits_max: 32 or 64 = widest key it must hold.  flags: OR of HCC_PIPELINE_*. */
#define HCC_PIPELINE_HOST_STAGING 1u
#define HCC_PIPELINE_PAIR 2u
HCC_API int32_t hcc_pipeline_create(uint64_t n_max, uint32_t container_bits_max, uint32_t flags,
                            hcc_pipeline **out);
HCC_API int32_t hcc_pipeline_destroy(hcc_pipeline *p);
/* Low key bits the pipeline's sort leaves unordered (hcc_sort_range's bit_lo);
 * 0 = the full sort (default).  Values above the key's used bits mean "do not sort at all". */
HCC_API int32_t hcc_pipeline_set_sort_skip_bits(hcc_pipeline *p, uint32_t bits);

/* Enqueue encode + sort + trace of one batch on `stream` (device pointers).
 *  order HCC_ORDER_HCC:      keys = hcc_encode(rays, cut);               `cut` required
 *  order HCC_ORDER_TWOPOINT: keys = hcc_encode_twopoint(rays, root box, key_bits); cut ignored
 *  order HCC_ORDER_NOSORT:   no keys, no sort; rays traced in input order
 * then perm = hcc_sort(keys) and hcc_trace(bvh, rays, perm, mode, hits_dev).
 * perm_out_dev: NULL, or uint32[n] that receives the permutation (untouched for NOSORT).
 * key_bits is used by TWOPOINT only. */
HCC_API int32_t hcc_reorder_trace(hcc_pipeline *p, const hcc_bvh *bvh, const hcc_cut *cut, int32_t order,
                          uint32_t key_bits, const float *rays_dev, uint64_t n, int32_t mode,
                          void *hits_dev, uint32_t *perm_out_dev, void *stream);
/* The same with HOST buffers: copies rays_host (32 n bytes; pinned memory makes the copy
 * asynchronous) to the device, runs the batch, copies the hits (16 n bytes CLOSEST, n bytes
 * ANY) to hits_host and synchronises `stream` before returning.  Needs HCC_PIPELINE_HOST_STAGING. */
HCC_API int32_t hcc_reorder_trace_host(hcc_pipeline *p, const hcc_bvh *bvh, const hcc_cut *cut, int32_t order,
                               uint32_t key_bits, const float *rays_host, uint64_t n, int32_t mode,
                               void *hits_host, void *stream);
/* The same without the final synchronisation: the call only enqueues on `stream` (the copies are
 * asynchronous if the host buffers are pinned); hits_host is valid after hcc_pipeline_synchronize
 * (or a synchronisation of `stream`).  Two pipelines on two streams overlap one batch's copies with
 * the other batch's kernels. */
HCC_API int32_t hcc_reorder_trace_host_async(hcc_pipeline *p, const hcc_bvh *bvh, const hcc_cut *cut, int32_t order,
                                     uint32_t key_bits, const float *rays_host, uint64_t n, int32_t mode,
                                     void *hits_host, void *stream);
/* Both batches of one bounce in one call: batch a (say the diffuse rays, HCC_TRACE_CLOSEST) and batch b (the
 * shadow rays, HCC_TRACE_ANY) go through the same three kernels as in hcc_reorder_trace, scheduled so that they
 * fill each other's gaps: up to 2^23 rays in total, b's keys and sort run on a stream of the pipeline's own beside a's (forked from and
 * joined back into `stream` by events), then a's traversal kernel and, as a dependent launch that does not wait
 * for it, b's: b's CTAs become resident as a's run out.  Both batches must be complete in memory when the call
 * is made.  Results are those of two hcc_reorder_trace calls.  Either n may be 0.  Needs a pipeline created
 * with HCC_PIPELINE_PAIR (else HCC_ERR_INVALID_ARG).  Per-stage timing is not recorded. */
HCC_API int32_t hcc_reorder_trace_pair(hcc_pipeline *p, const hcc_bvh *bvh, const hcc_cut *cut, int32_t order,
                               uint32_t key_bits, const float *rays_a_dev, uint64_t n_a, int32_t mode_a,
                               void *hits_a_dev, const float *rays_b_dev, uint64_t n_b, int32_t mode_b,
                               void *hits_b_dev, void *stream);
/* Waits until the pipeline's last enqueued call has finished. */
HCC_API int32_t hcc_pipeline_synchronize(hcc_pipeline *p);
/* Per-stage timing: with enable != 0 every later hcc_reorder_trace(_host) call records CUDA events on its
 * stream between the stages (this orders the stages completely: no kernel of a call overlaps the next one's
 * prologue).  Off by default. */
HCC_API int32_t hcc_pipeline_set_timing(hcc_pipeline *p, uint32_t enable);
/* Device time of the stages of the pipeline's last timed call: ms[0] encode, [1] sort, [2] trace,
 * [3] host->device copy, [4] device->host copy (3, 4 = 0 for the device form).  Waits for that call to
 * finish.  HCC_ERR_INVALID_ARG if the last call was not timed (hcc_pipeline_set_timing). */
HCC_API int32_t hcc_pipeline_stage_ms(hcc_pipeline *p, float ms[5]);

/* ANC, "average number of codes per warp" (Table 7): for every group of 32
 * consecutive ranks j (the rays one traversal warp holds) the number of distinct keys
 * keys_dev[perm_dev[j]] (perm_dev NULL = identity).  out_dev = uint64[2], zeroed by the call:
 * [0] = sum over warps of distinct keys, [1] = number of warps.  keys_dev is in ORIGINAL ray
 * order (hcc_sort clobbers its input: pass a copy made before sorting). */
HCC_API int32_t hcc_anc(const void *keys_dev, const uint32_t *perm_dev, uint64_t n, uint32_t container_bits,
                uint64_t *out_dev, void *stream);

#ifdef __cplusplus
}
#endif
#endif /* HCC_H */
