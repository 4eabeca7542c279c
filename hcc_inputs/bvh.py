"""ctypes front end of the host binned-SAH builder (bvh_builder.c)."""
import ctypes

import numpy as np

from . import build as _build

NODE_DTYPE = np.dtype([("lo", np.float32, 3), ("hi", np.float32, 3),
                       ("left_or_first", np.uint32), ("count", np.uint32)])
assert NODE_DTYPE.itemsize == 32

_lib = None


def _load():
    global _lib
    if _lib is None:
        _lib = ctypes.CDLL(_build.build())
        _lib.hcc_build_bvh.restype = ctypes.c_int
        _lib.hcc_build_bvh.argtypes = [ctypes.c_void_p, ctypes.c_uint32, ctypes.c_uint32, ctypes.c_uint32,
                                       ctypes.c_void_p, ctypes.c_void_p, ctypes.c_void_p, ctypes.c_void_p]
    return _lib


class BVH:
    """Canonical binary BVH: `nodes` (NODE_DTYPE [n_nodes]), `prim_idx` (uint32 [n_tris]),
    `tris` (float32 [n_tris,3,3], caller order; a leaf's triangles are
    tris[prim_idx[first:first+count]])."""

    def __init__(self, nodes, prim_idx, tris, max_depth):
        self.nodes, self.prim_idx, self.tris, self.max_depth = nodes, prim_idx, tris, int(max_depth)

    @property
    def n_nodes(self):
        return int(self.nodes.shape[0])

    @property
    def n_tris(self):
        return int(self.tris.shape[0])

    @property
    def n_leaves(self):
        return int((self.nodes["count"] > 0).sum())


def build_bvh(tris, max_leaf=4, n_bins=16):
    tris = np.ascontiguousarray(tris, dtype=np.float32).reshape(-1, 3, 3)
    n = tris.shape[0]
    if n == 0:
        raise ValueError("empty scene")
    nodes = np.zeros(2 * n, dtype=NODE_DTYPE)
    prim_idx = np.zeros(n, dtype=np.uint32)
    n_nodes = ctypes.c_uint32(0)
    max_depth = ctypes.c_uint32(0)
    rc = _load().hcc_build_bvh(tris.ctypes.data, n, max_leaf, n_bins, nodes.ctypes.data,
                               prim_idx.ctypes.data, ctypes.byref(n_nodes), ctypes.byref(max_depth))
    if rc != 0:
        raise RuntimeError(f"hcc_build_bvh failed: {rc}")
    return BVH(np.ascontiguousarray(nodes[:n_nodes.value]), prim_idx, tris, max_depth.value)


def make_bvh(nodes_list, tris, prim_idx=None):
    """Hand-built BVH for tests: nodes_list = [(lo, hi, left_or_first, count), ...]."""
    nodes = np.zeros(len(nodes_list), dtype=NODE_DTYPE)
    for i, (lo, hi, lf, c) in enumerate(nodes_list):
        nodes[i] = (np.asarray(lo, np.float32), np.asarray(hi, np.float32), lf, c)
    tris = np.ascontiguousarray(tris, dtype=np.float32).reshape(-1, 3, 3)
    if prim_idx is None:
        prim_idx = np.arange(tris.shape[0], dtype=np.uint32)
    depth = np.zeros(len(nodes_list), dtype=np.int64)
    for i in range(len(nodes_list)):
        if nodes["count"][i] == 0:
            l = int(nodes["left_or_first"][i])
            depth[l] = depth[l + 1] = depth[i] + 1
    return BVH(nodes, np.ascontiguousarray(prim_idx, dtype=np.uint32), tris, depth.max())
