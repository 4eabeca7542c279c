"""Python binding of libhcc_b200.so — the B200-native hot path of "Faster Ray Tracing
through Hierarchy Cut Code" (arxiv 2305.16652): density + cut selection, key
computation, radix sort of ray ids, BVH traversal of the reordered rays.

Argument marshalling only.  Every step runs in the CUDA kernels behind the C ABI of
include/hcc.h; the functions here carry the same names without the `hcc_` prefix.
torch supplies device memory and streams, nothing else.  There is no CPU fallback: a
missing library raises at import.
"""
import ctypes
import os

import numpy as np
import torch

_HERE = os.path.dirname(os.path.abspath(__file__))
# HCC_B200_LIB names another build of the same library (kernel tuning variants); default: the in-tree one
LIB_PATH = os.environ.get("HCC_B200_LIB") or os.path.join(_HERE, "libhcc_b200.so")

MISS_PRIM = 0xFFFFFFFF
MAX_LEVELS = 16
TRACE_CLOSEST, TRACE_ANY = 0, 1

_vp, _u32, _u64, _i32 = ctypes.c_void_p, ctypes.c_uint32, ctypes.c_uint64, ctypes.c_int32
_f32 = ctypes.c_float
_pu32, _pu64 = ctypes.POINTER(ctypes.c_uint32), ctypes.POINTER(ctypes.c_uint64)

# name -> argtypes; every function returns int32 status except the two noted below
_SIGNATURES = {
    "hcc_bvh_create": [_vp, _u32, _vp, _u32, _vp, _vp, ctypes.POINTER(_vp)],
    "hcc_bvh_destroy": [_vp],
    "hcc_bvh_info": [_vp, _pu32, _pu32, _pu32, _pu32, _vp, _vp],
    "hcc_density": [_vp, _f32, _vp, _vp],
    "hcc_cut_create": [_u32, ctypes.POINTER(_vp)],
    "hcc_cut_destroy": [_vp],
    "hcc_select_cut": [_vp, _vp, _u32, _u32, _vp, _vp],
    "hcc_select_cut_levels": [_vp, _vp, _vp, _u32, _u32, _vp, _vp],
    "hcc_select_cut_levels_ex": [_vp, _vp, _vp, _u32, _u32, _u32, _vp, _vp],
    "hcc_cut_info": [_vp, _pu32, _pu32, _pu32, _pu32, _pu32, _pu64, _pu64],
    "hcc_cut_read": [_vp, _vp, _vp, _vp],
    "hcc_select_cut_flat_workspace_bytes": [_vp, _u32, _pu64],
    "hcc_select_cut_flat": [_vp, _vp, _u32, _vp, _vp, _vp, _u64, _vp],
    "hcc_encode": [_vp, _u64, _vp, _vp, _vp],
    "hcc_encode_twopoint": [_vp, _u64, _vp, _vp, _u32, _vp, _vp],
    "hcc_sort_workspace_bytes": [_u64, _u32, _pu64],
    "hcc_sort": [_vp, _u64, _u32, _u32, _vp, _vp, _u64, _vp],
    "hcc_sort_static": [_vp, _u64, _u32, _u32, _vp, _vp],
    "hcc_encode_ppc": [_vp, _vp, _u64, _u32, _vp, _vp],
    "hcc_select_grid": [_vp, _vp, _u32, _u32, _vp, _vp],
    "hcc_cut_read_boxes": [_vp, _vp, _vp],
    "hcc_sort_range": [_vp, _u64, _u32, _u32, _u32, _vp, _vp, _u64, _vp],
    "hcc_pipeline_set_sort_skip_bits": [_vp, _u32],
    "hcc_trace": [_vp, _vp, _u64, _vp, _i32, _vp, _vp],
    "hcc_pipeline_create": [_u64, _u32, _u32, ctypes.POINTER(_vp)],
    "hcc_pipeline_destroy": [_vp],
    "hcc_reorder_trace": [_vp, _vp, _vp, _i32, _u32, _vp, _u64, _i32, _vp, _vp, _vp],
    "hcc_reorder_trace_host": [_vp, _vp, _vp, _i32, _u32, _vp, _u64, _i32, _vp, _vp],
    "hcc_reorder_trace_host_async": [_vp, _vp, _vp, _i32, _u32, _vp, _u64, _i32, _vp, _vp],
    "hcc_reorder_trace_pair": [_vp, _vp, _vp, _i32, _u32, _vp, _u64, _i32, _vp, _vp, _u64, _i32, _vp, _vp],
    "hcc_pipeline_set_timing": [_vp, _u32],
    "hcc_pipeline_synchronize": [_vp],
    "hcc_pipeline_stage_ms": [_vp, _vp],
    "hcc_trace_stats": [_vp, _vp, _u64, _vp, _i32, _vp, _vp, _vp],
    "hcc_anc": [_vp, _vp, _u64, _u32, _vp, _vp],
}
EXPORTS = sorted(list(_SIGNATURES) + ["hcc_last_error", "hcc_version"])

ORDER_NOSORT, ORDER_TWOPOINT, ORDER_HCC = 0, 1, 2

_lib = None


def lib():
    """The loaded C-ABI library.  Raises if it has not been built (no fallback)."""
    global _lib
    if _lib is None:
        if not os.path.exists(LIB_PATH):
            raise ImportError(
                f"{LIB_PATH} is missing: build it with `python -m paper_2305_16652_b200.build` "
                "(or __graft_entry__.build()).  There is no CPU fallback.")
        L = ctypes.CDLL(LIB_PATH)
        for name, args in _SIGNATURES.items():
            fn = getattr(L, name)
            fn.argtypes = args
            fn.restype = _i32
        L.hcc_last_error.argtypes = []
        L.hcc_last_error.restype = ctypes.c_char_p
        L.hcc_version.argtypes = []
        L.hcc_version.restype = _i32
        _lib = L
    return _lib


class HccError(RuntimeError):
    def __init__(self, status, message):
        super().__init__(f"hcc status {status}: {message}")
        self.status = status


def _check(rc):
    if rc != 0:
        raise HccError(rc, lib().hcc_last_error().decode("utf-8", "replace"))


def _stream(stream=None):
    s = torch.cuda.current_stream() if stream is None else stream
    return _vp(s.cuda_stream)


def _dev(t, dtypes, what):
    if not (isinstance(t, torch.Tensor) and t.is_cuda and t.is_contiguous() and t.dtype in dtypes):
        raise TypeError(f"{what}: expected a contiguous CUDA tensor of dtype in {dtypes}")
    return _vp(t.data_ptr())


def version():
    return int(lib().hcc_version())


# ---------------------------------------------------------------------------------- BVH
class Bvh:
    """Device BVH handle (hcc_bvh_create).  nodes: numpy structured array of 32-byte
    canonical nodes; tris: float32 [n,3,3]; prim_idx: uint32 [n] (all host)."""

    def __init__(self, nodes, tris, prim_idx, stream=None):
        nodes = np.ascontiguousarray(nodes)
        if nodes.dtype.itemsize != 32:
            raise TypeError("nodes must be 32-byte canonical node records")
        tris = np.ascontiguousarray(tris, dtype=np.float32).reshape(-1, 9)
        prim_idx = np.ascontiguousarray(prim_idx, dtype=np.uint32)
        if prim_idx.shape[0] != tris.shape[0]:
            raise ValueError("prim_idx and tris disagree in length")
        self._h = _vp()
        _check(lib().hcc_bvh_create(nodes.ctypes.data, nodes.shape[0], tris.ctypes.data, tris.shape[0],
                                    prim_idx.ctypes.data, _stream(stream), ctypes.byref(self._h)))
        a = [_u32() for _ in range(4)]
        lo, hi = (ctypes.c_float * 3)(), (ctypes.c_float * 3)()
        _check(lib().hcc_bvh_info(self._h, *[ctypes.byref(x) for x in a], lo, hi))
        self.n_nodes, self.n_tris, self.n_leaves, self.max_depth = [int(x.value) for x in a]
        self.scene_lo = np.array(list(lo), dtype=np.float32)
        self.scene_hi = np.array(list(hi), dtype=np.float32)

    def close(self):
        if getattr(self, "_h", None) is not None and self._h and _lib is not None:   # _lib is None at interpreter exit
            _lib.hcc_bvh_destroy(self._h)
            self._h = None

    __del__ = close


def bvh_create(nodes, tris, prim_idx, stream=None):
    return Bvh(nodes, tris, prim_idx, stream)


# ---------------------------------------------------------------------------------- (a1)
def density(bvh, lam=0.125, out=None, stream=None):
    """hcc_density: float32 CUDA tensor [n_nodes] (Eq. 1)."""
    if out is None:
        out = torch.empty(bvh.n_nodes, dtype=torch.float32, device="cuda")
    _check(lib().hcc_density(bvh._h, float(lam), _dev(out, (torch.float32,), "density"), _stream(stream)))
    return out


class Cut:
    """Device level tables of one cut hierarchy (hcc_cut_create / hcc_select_cut)."""

    def __init__(self, max_K):
        self._h = _vp()
        self.max_K = int(max_K)
        _check(lib().hcc_cut_create(self.max_K, ctypes.byref(self._h)))

    def info(self):
        m, K_eff, bits, cont = _u32(), _u32(), _u32(), _u32()
        w = (_u32 * MAX_LEVELS)()
        ne, nt = _u64(), _u64()
        _check(lib().hcc_cut_info(self._h, ctypes.byref(m), w, ctypes.byref(K_eff), ctypes.byref(bits),
                                  ctypes.byref(cont), ctypes.byref(ne), ctypes.byref(nt)))
        return dict(m=int(m.value), widths=[int(w[i]) for i in range(m.value)], K_eff=int(K_eff.value),
                    bits_used=int(bits.value), container_bits=int(cont.value),
                    n_entries=int(ne.value), n_tables=int(nt.value))

    def read(self, stream=None):
        """(entry_node uint32 [n_entries], table_cnt uint32 [n_tables]) on the host."""
        i = self.info()
        ent = np.empty(i["n_entries"], dtype=np.uint32)
        cnt = np.empty(i["n_tables"], dtype=np.uint32)
        _check(lib().hcc_cut_read(self._h, ent.ctypes.data, cnt.ctypes.data, _stream(stream)))
        return ent, cnt

    def read_boxes(self, stream=None):
        """hcc_cut_read_boxes: float32 [n_entries, 6] (lo.xyz, hi.xyz) on the host."""
        boxes = np.empty((self.info()["n_entries"], 6), dtype=np.float32)
        _check(lib().hcc_cut_read_boxes(self._h, boxes.ctypes.data, _stream(stream)))
        return boxes

    def close(self):
        if getattr(self, "_h", None) is not None and self._h and _lib is not None:   # _lib is None at interpreter exit
            _lib.hcc_cut_destroy(self._h)
            self._h = None

    __del__ = close


def select_cut(bvh, density_dev, K, key_bits, cut=None, stream=None):
    """hcc_select_cut (Alg. 2 / Alg. 3 level tables)."""
    if cut is None:
        cut = Cut(max(int(K), 64))
    _check(lib().hcc_select_cut(bvh._h, _dev(density_dev, (torch.float32,), "density"), int(K), int(key_bits),
                                cut._h, _stream(stream)))
    return cut


CUT_ALG3_DISCARD = 1


def select_cut_levels(bvh, density_dev, widths, key_bits, cut=None, stream=None, flags=0):
    """hcc_select_cut_levels(_ex): level tables of explicit widths; flags=CUT_ALG3_DISCARD builds the upper
    levels by Algorithm 3 as printed."""
    w = np.ascontiguousarray(widths, dtype=np.uint32)
    if cut is None:
        cut = Cut(max(int(np.prod(w.astype(np.int64))), 64))
    _check(lib().hcc_select_cut_levels_ex(bvh._h, _dev(density_dev, (torch.float32,), "density"), w.ctypes.data,
                                          w.shape[0], int(key_bits), int(flags), cut._h, _stream(stream)))
    return cut


def select_grid(bvh, widths, key_bits, cut=None, stream=None):
    """hcc_select_grid (f4): level tables whose entries are regular grid cells."""
    w = np.ascontiguousarray(widths, dtype=np.uint32)
    if cut is None:
        cut = Cut(max(int(np.prod(w.astype(np.int64))), 64))
    _check(lib().hcc_select_grid(bvh._h, w.ctypes.data, w.shape[0], int(key_bits), cut._h, _stream(stream)))
    return cut


def select_cut_flat(bvh, density_dev, K, stream=None):
    """hcc_select_cut_flat: Alg. 2 for any K.  Returns (cut_nodes int32 CUDA [K] viewed as
    uint32 bits, count CUDA int32 [1])."""
    need = _u64()
    _check(lib().hcc_select_cut_flat_workspace_bytes(bvh._h, int(K), ctypes.byref(need)))
    ws = torch.empty(int(need.value), dtype=torch.uint8, device="cuda")
    out = torch.empty(int(K), dtype=torch.int32, device="cuda")
    cnt = torch.zeros(4, dtype=torch.int32, device="cuda")
    _check(lib().hcc_select_cut_flat(bvh._h, _dev(density_dev, (torch.float32,), "density"), int(K),
                                     _vp(out.data_ptr()), _vp(cnt.data_ptr()), _vp(ws.data_ptr()),
                                     int(need.value), _stream(stream)))
    return out, cnt


# ---------------------------------------------------------------------------------- (a2)
def _key_dtype(container_bits):
    return torch.int32 if container_bits == 32 else torch.int64


def _rays_dev(rays):
    if not (isinstance(rays, torch.Tensor) and rays.is_cuda and rays.is_contiguous()
            and rays.dtype == torch.float32 and rays.dim() == 2 and rays.shape[1] == 8):
        raise TypeError("rays: expected a contiguous float32 CUDA tensor [n, 8]")
    return _vp(rays.data_ptr())


def encode(rays, cut, keys=None, stream=None):
    """hcc_encode: keys as an int32 / int64 CUDA tensor holding the uint32 / uint64 bits."""
    n = rays.shape[0]
    dt = _key_dtype(cut.info()["container_bits"])
    if keys is None:
        keys = torch.empty(n, dtype=dt, device="cuda")
    _check(lib().hcc_encode(_rays_dev(rays), n, cut._h, _dev(keys, (dt,), "keys"), _stream(stream)))
    return keys


def encode_twopoint(rays, scene_lo, scene_hi, key_bits, keys=None, stream=None):
    n = rays.shape[0]
    dt = _key_dtype(32 if key_bits <= 32 else 64)
    if keys is None:
        keys = torch.empty(n, dtype=dt, device="cuda")
    lo = (ctypes.c_float * 3)(*[float(x) for x in scene_lo])
    hi = (ctypes.c_float * 3)(*[float(x) for x in scene_hi])
    _check(lib().hcc_encode_twopoint(_rays_dev(rays), n, lo, hi, int(key_bits), _dev(keys, (dt,), "keys"),
                                     _stream(stream)))
    return keys


def encode_ppc(bvh, rays, key_bits, keys=None, stream=None):
    """hcc_encode_ppc (f3): prefix path code of every ray."""
    n = rays.shape[0]
    dt = _key_dtype(32 if key_bits <= 32 else 64)
    if keys is None:
        keys = torch.empty(n, dtype=dt, device="cuda")
    _check(lib().hcc_encode_ppc(bvh._h, _rays_dev(rays), n, int(key_bits), _dev(keys, (dt,), "keys"), _stream(stream)))
    return keys


# ---------------------------------------------------------------------------------- (a3)
def sort_workspace_bytes(n, container_bits):
    need = _u64()
    _check(lib().hcc_sort_workspace_bytes(int(n), int(container_bits), ctypes.byref(need)))
    return int(need.value)


def sort(keys, bits_used, perm=None, workspace=None, stream=None, bit_lo=0):
    """hcc_sort / hcc_sort_range: stable ascending permutation of ray ids (int32 CUDA [n]) by the key
    bits [bit_lo, bits_used).  keys is clobbered."""
    n = keys.shape[0]
    cb = 32 if keys.dtype == torch.int32 else 64
    if perm is None:
        perm = torch.empty(n, dtype=torch.int32, device="cuda")
    if workspace is None:
        workspace = torch.empty(sort_workspace_bytes(n, cb), dtype=torch.uint8, device="cuda")
    _check(lib().hcc_sort_range(_dev(keys, (torch.int32, torch.int64), "keys"), n, cb, int(bit_lo), int(bits_used),
                                _dev(perm, (torch.int32,), "perm"), _vp(workspace.data_ptr()), workspace.numel(),
                                _stream(stream)))
    return perm


SORT_STATIC_MAX_N = 262144


def sort_static(keys, bits_used, perm, stream=None):
    """hcc_sort_static: hcc_sort without a workspace argument, for code that runs where device memory cannot be
    allocated (a plug-in inside an application that owns the GPU's memory, a render loop that must stay off the
    driver's allocation lock).  The workspace is a 4 MiB array inside the library, one per GPU, shared by all
    calls: at most SORT_STATIC_MAX_N pairs, and two calls must not run on the GPU at the same time.  `perm`
    (int32 CUDA [n]) is the caller's, as are the keys (clobbered): this function creates no tensor."""
    n = keys.shape[0]
    cb = 32 if keys.dtype == torch.int32 else 64
    _check(lib().hcc_sort_static(_dev(keys, (torch.int32, torch.int64), "keys"), n, cb, int(bits_used),
                                 _dev(perm, (torch.int32,), "perm"), _stream(stream)))
    return perm


# ---------------------------------------------------------------------------------- (a4)
def trace(bvh, rays, perm=None, mode=TRACE_CLOSEST, hits=None, stream=None):
    """hcc_trace.  CLOSEST: float32 CUDA [n,4] = (t, prim bits, u, v); ANY: uint8 CUDA [n]."""
    n = rays.shape[0]
    if hits is None:
        hits = (torch.empty((n, 4), dtype=torch.float32, device="cuda") if mode == TRACE_CLOSEST
                else torch.empty(n, dtype=torch.uint8, device="cuda"))
    p = _vp(0) if perm is None else _dev(perm, (torch.int32,), "perm")
    _check(lib().hcc_trace(bvh._h, _rays_dev(rays), n, p, int(mode), _vp(hits.data_ptr()), _stream(stream)))
    return hits


def hits_to_numpy(hits):
    """(t float32 [n], prim uint32 [n], u, v) from a CLOSEST hits tensor."""
    h = hits.detach().cpu().numpy()
    return h[:, 0].copy(), h[:, 1].copy().view(np.uint32), h[:, 2].copy(), h[:, 3].copy()


def keys_to_numpy(keys):
    """uint64 numpy array of the key bits."""
    k = keys.detach().cpu().numpy()
    return (k.view(np.uint32) if k.dtype == np.int32 else k.view(np.uint64)).astype(np.uint64)


def trace_stats(bvh, rays, perm=None, mode=TRACE_CLOSEST, stream=None):
    """hcc_trace_stats: dict(nodes, tris, rays, max_stack, node_bytes_per_ray, tri_bytes_per_ray; per warp-level
    node step: distinct node records (records_per_step) and lanes taking part (lanes_per_step); per warp-level
    triangle round: triangle tests (tri_tests_per_round; a lane can test several triangles of its leaf in one round))."""
    n = rays.shape[0]
    hits = (torch.empty((n, 4), dtype=torch.float32, device="cuda") if mode == TRACE_CLOSEST
            else torch.empty(n, dtype=torch.uint8, device="cuda"))
    st = torch.zeros(8, dtype=torch.int64, device="cuda")
    p = _vp(0) if perm is None else _dev(perm, (torch.int32,), "perm")
    _check(lib().hcc_trace_stats(bvh._h, _rays_dev(rays), n, p, int(mode), _vp(hits.data_ptr()),
                                 _vp(st.data_ptr()), _stream(stream)))
    nodes, tris, nr, depth, records, steps, lanes, rounds = [int(x) for x in st.cpu().tolist()]
    return dict(nodes=nodes, tris=tris, rays=nr, max_stack=depth,
                node_bytes_per_ray=64.0 * nodes / max(nr, 1), tri_bytes_per_ray=64.0 * tris / max(nr, 1),
                warp_steps=steps, records_per_step=records / max(steps, 1), lanes_per_step=lanes / max(steps, 1),
                distinct_node_bytes_per_ray=64.0 * records / max(nr, 1),
                tri_rounds=rounds, tri_tests_per_round=tris / max(rounds, 1))


def anc(keys, perm=None, stream=None):
    """hcc_anc: average number of distinct codes per 32-ray warp."""
    n = keys.shape[0]
    cb = 32 if keys.dtype == torch.int32 else 64
    out = torch.zeros(2, dtype=torch.int64, device="cuda")
    p = _vp(0) if perm is None else _dev(perm, (torch.int32,), "perm")
    _check(lib().hcc_anc(_dev(keys, (torch.int32, torch.int64), "keys"), p, n, cb, _vp(out.data_ptr()),
                         _stream(stream)))
    s, w = [int(x) for x in out.cpu().tolist()]
    return s / max(w, 1)


# ---------------------------------------------------------------------------------- pipeline
class Pipeline:
    """Per-batch scratch (hcc_pipeline_create) and the one-call path encode -> sort -> trace.  host_staging: scratch for the
    host-buffer calls; pair: scratch for reorder_trace_pair."""

    def __init__(self, n_max, container_bits_max=64, host_staging=False, pair=False):
        self._h = _vp()
        self.n_max = int(n_max)
        _check(lib().hcc_pipeline_create(self.n_max, int(container_bits_max), (1 if host_staging else 0) | (2 if pair else 0),
                                         ctypes.byref(self._h)))

    def set_sort_skip_bits(self, bits):
        """hcc_pipeline_set_sort_skip_bits: low key bits the sort leaves unordered."""
        _check(lib().hcc_pipeline_set_sort_skip_bits(self._h, int(bits)))

    def reorder_trace(self, bvh, cut, order, rays, mode=TRACE_CLOSEST, hits=None, key_bits=32,
                      perm_out=None, stream=None):
        """hcc_reorder_trace on device tensors.  Returns hits."""
        n = rays.shape[0]
        if hits is None:
            hits = (torch.empty((n, 4), dtype=torch.float32, device="cuda") if mode == TRACE_CLOSEST
                    else torch.empty(n, dtype=torch.uint8, device="cuda"))
        po = _vp(0) if perm_out is None else _dev(perm_out, (torch.int32,), "perm_out")
        _check(lib().hcc_reorder_trace(self._h, bvh._h, _vp(0) if cut is None else cut._h, int(order),
                                       int(key_bits), _rays_dev(rays), n, int(mode), _vp(hits.data_ptr()), po,
                                       _stream(stream)))
        return hits

    def reorder_trace_pair(self, bvh, cut, order, rays_a, mode_a, hits_a, rays_b, mode_b, hits_b, key_bits=32, stream=None):
        """hcc_reorder_trace_pair: both batches of one bounce in one call (b's keys and sort overlap a's traversal)."""
        _check(lib().hcc_reorder_trace_pair(self._h, bvh._h, _vp(0) if cut is None else cut._h, int(order), int(key_bits),
                                            _rays_dev(rays_a), rays_a.shape[0], int(mode_a), _vp(hits_a.data_ptr()),
                                            _rays_dev(rays_b), rays_b.shape[0], int(mode_b), _vp(hits_b.data_ptr()),
                                            _stream(stream)))
        return hits_a, hits_b

    def set_timing(self, enable=True):
        """hcc_pipeline_set_timing: record the per-stage events of later calls (stage_ms)."""
        _check(lib().hcc_pipeline_set_timing(self._h, 1 if enable else 0))

    def reorder_trace_host(self, bvh, cut, order, rays_host, hits_host, mode=TRACE_CLOSEST, key_bits=32,
                           stream=None):
        """hcc_reorder_trace_host: rays_host / hits_host are HOST tensors or numpy arrays
        (pin them for asynchronous copies).  Synchronises before returning."""
        n = rays_host.shape[0]
        rp = rays_host.data_ptr() if isinstance(rays_host, torch.Tensor) else rays_host.ctypes.data
        hp = hits_host.data_ptr() if isinstance(hits_host, torch.Tensor) else hits_host.ctypes.data
        _check(lib().hcc_reorder_trace_host(self._h, bvh._h, _vp(0) if cut is None else cut._h, int(order),
                                            int(key_bits), _vp(rp), n, int(mode), _vp(hp), _stream(stream)))
        return hits_host

    def reorder_trace_host_async(self, bvh, cut, order, rays_host, hits_host, mode=TRACE_CLOSEST, key_bits=32,
                                 stream=None):
        """hcc_reorder_trace_host_async: enqueue only; hits_host is valid after synchronize()."""
        n = rays_host.shape[0]
        rp = rays_host.data_ptr() if isinstance(rays_host, torch.Tensor) else rays_host.ctypes.data
        hp = hits_host.data_ptr() if isinstance(hits_host, torch.Tensor) else hits_host.ctypes.data
        _check(lib().hcc_reorder_trace_host_async(self._h, bvh._h, _vp(0) if cut is None else cut._h, int(order),
                                                  int(key_bits), _vp(rp), n, int(mode), _vp(hp), _stream(stream)))
        return hits_host

    def synchronize(self):
        """hcc_pipeline_synchronize: wait for the pipeline's last enqueued call."""
        _check(lib().hcc_pipeline_synchronize(self._h))

    def stage_ms(self):
        """dict(encode, sort, trace, h2d, d2h) in ms for the last call (waits for it)."""
        ms = (ctypes.c_float * 5)()
        _check(lib().hcc_pipeline_stage_ms(self._h, ms))
        return dict(encode=ms[0], sort=ms[1], trace=ms[2], h2d=ms[3], d2h=ms[4])

    def close(self):
        if getattr(self, "_h", None) is not None and self._h and _lib is not None:   # _lib is None at interpreter exit
            _lib.hcc_pipeline_destroy(self._h)
            self._h = None

    __del__ = close
