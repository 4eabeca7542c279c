"""ORACLE — TEST INFRASTRUCTURE ONLY (see hcc_oracle.c's header).

numpy front end of oracle/liboracle.so plus the host-side rules that are not
arithmetic (the level-width rule R-ML).  Only tests/, __graft_entry__.smoke() and
bench.py's cpu_baseline / --impl reference legs may import this package; the
product (paper_2305_16652_b200/) never does, and this package never imports it.

Arrays: nodes = structured array of 32-byte canonical nodes (lo[3], hi[3],
left_or_first, count); rays = float32 [n,8] (o, tmin, d, tmax); tris = float32 [N,3,3].
"""
import ctypes

import numpy as np

from . import build as _build

INVALID = 0xFFFFFFFF
_lib = None
_vp = ctypes.c_void_p
_u32 = ctypes.c_uint32
_u64 = ctypes.c_uint64


def _load():
    global _lib
    if _lib is None:
        L = ctypes.CDLL(_build.build())
        L.oracle_had.argtypes = [_vp, _u32, ctypes.c_float, _vp]
        L.oracle_had.restype = None
        L.oracle_subtree_leaves.argtypes = [_vp, _u32, _vp]
        L.oracle_subtree_leaves.restype = None
        L.oracle_cut.argtypes = [_vp, _vp, _vp, _u32, _u32, _u32, _vp]
        L.oracle_cut.restype = _u32
        L.oracle_level_tables.argtypes = [_vp, _vp, _vp, _vp, _u32, _vp, _vp]
        L.oracle_level_tables.restype = None
        L.oracle_level_tables_ex.argtypes = [_vp, _vp, _vp, _vp, _u32, ctypes.c_int, _vp, _vp]
        L.oracle_level_tables_ex.restype = None
        L.oracle_cut_ex.argtypes = [_vp, _vp, _vp, _u32, _u32, _u32, ctypes.c_int, _vp]
        L.oracle_cut_ex.restype = _u32
        L.oracle_slab_hit.argtypes = [_vp, _vp, _vp]
        L.oracle_slab_hit.restype = ctypes.c_int
        L.oracle_encode_hcc.argtypes = [_vp, _u64, _vp, _vp, _u32, _vp, _vp, _vp]
        L.oracle_encode_hcc.restype = None
        L.oracle_encode_twopoint.argtypes = [_vp, _u64, _vp, _vp, _u32, _vp]
        L.oracle_encode_twopoint.restype = None
        L.oracle_grid_tables.argtypes = [_vp, _vp, _vp, _u32, _vp]
        L.oracle_grid_tables.restype = None
        L.oracle_encode_tables.argtypes = [_vp, _u64, _vp, _vp, _u32, _vp, _vp]
        L.oracle_encode_tables.restype = None
        L.oracle_encode_ppc.argtypes = [_vp, _u64, _vp, _u32, _vp]
        L.oracle_encode_ppc.restype = ctypes.c_int
        L.oracle_sort_from_bit.argtypes = [_vp, _u64, _u32, _vp]
        L.oracle_sort_from_bit.restype = ctypes.c_int
        L.oracle_sort.argtypes = [_vp, _u64, _vp]
        L.oracle_sort.restype = ctypes.c_int
        L.oracle_tri_hit.argtypes = [_vp, _vp, _vp]
        L.oracle_tri_hit.restype = ctypes.c_int
        L.oracle_closest_brute.argtypes = [_vp, _u64, _vp, _u32, _vp, _vp, _vp, _vp]
        L.oracle_closest_brute.restype = None
        L.oracle_any_brute.argtypes = [_vp, _u64, _vp, _u32, _vp]
        L.oracle_any_brute.restype = None
        L.oracle_closest_bvh.argtypes = [_vp, _u64, _vp, _vp, _vp, _vp, _vp, _vp, _vp, _vp]
        L.oracle_closest_bvh.restype = ctypes.c_int
        L.oracle_any_bvh.argtypes = [_vp, _u64, _vp, _vp, _vp, _vp, _vp]
        L.oracle_any_bvh.restype = ctypes.c_int
        _lib = L
    return _lib


def _c(a, dtype=None):
    a = np.ascontiguousarray(a, dtype=dtype)
    return a


def _rays(rays):
    r = _c(rays, np.float32)
    assert r.ndim == 2 and r.shape[1] == 8
    return r


# --------------------------------------------------------------------------- (a1)
def had(nodes, lam=0.125):
    """Hierarchically accumulated density, Eq. 1.  float32 [n_nodes]."""
    nodes = _c(nodes)
    out = np.empty(nodes.shape[0], dtype=np.float32)
    _load().oracle_had(nodes.ctypes.data, nodes.shape[0], lam, out.ctypes.data)
    return out


def subtree_leaves(nodes):
    nodes = _c(nodes)
    out = np.empty(nodes.shape[0], dtype=np.uint32)
    _load().oracle_subtree_leaves(nodes.ctypes.data, nodes.shape[0], out.ctypes.data)
    return out


def cut(nodes, had_, K, start=0, need=2, leaves=None, discard=False):
    """Cut(start, K, need): Algorithm 2 from `start`; need > 2 gives
    Algorithm 3's "large enough subtree" test; discard=True is the literal Algorithm 3 (a node
    that is not large enough is dropped).  Node ids, HAD-descending (:192)."""
    nodes = _c(nodes)
    had_ = _c(had_, np.float32)
    if leaves is None:
        leaves = subtree_leaves(nodes)
    leaves = _c(leaves, np.uint32)
    out = np.empty(max(int(K), 1), dtype=np.uint32)
    n = _load().oracle_cut_ex(nodes.ctypes.data, had_.ctypes.data, leaves.ctypes.data,
                              int(start), int(K), int(need), 1 if discard else 0, out.ctypes.data)
    return out[:n].copy()


def level_widths(K, key_bits):
    """Reading R-ML: how a (K, B) request maps onto the
    paper's encoders.  Returns (widths, K_eff).
      K <= B            -> one level of K entries: plain HCC
      otherwise         -> the fewest levels m >= 2 whose power-of-two widths, exponents of
                           K = 2^k split as evenly as possible (larger first), satisfy
                           sum(w) <= B; if no m works k is reduced.  K = (B/2)^2 gives the
                           paper's two-level MLHCC."""
    K, B = int(K), int(key_bits)
    if K < 1 or B < 1:
        raise ValueError("K and key_bits must be positive")
    if K <= B:
        return [K], K
    k = K.bit_length() - 1           # floor(log2 K)
    while k >= 1:
        for m in range(2, k + 1):
            q, r = divmod(k, m)
            w = [1 << (q + 1)] * r + [1 << q] * (m - r)
            if sum(w) <= B:
                return w, 1 << k
        k -= 1
    return [min(K, B)], min(K, B)


class Tables:
    """Level tables of one cut hierarchy (oracle_level_tables)."""

    def __init__(self, widths, entry_node, table_cnt):
        self.widths = [int(w) for w in widths]
        self.entry_node, self.table_cnt = entry_node, table_cnt
        self.ent_off, self.tab_off, self.n_tables = [], [], []
        e = t = 0
        nt = 1
        for w in self.widths:
            self.ent_off.append(e); self.tab_off.append(t); self.n_tables.append(nt)
            e += nt * w; t += nt; nt *= w
        self.bits_used = sum(self.widths)

    def table(self, level, t):
        w = self.widths[level]
        c = int(self.table_cnt[self.tab_off[level] + t])
        o = self.ent_off[level] + t * w
        return self.entry_node[o:o + c]

    def level_entries(self, level):
        w = self.widths[level]
        o = self.ent_off[level]
        return self.entry_node[o:o + self.n_tables[level] * w]

    def finest_cut(self):
        """Node ids of all valid last-level entries: "the final cut nodes"."""
        e = self.level_entries(len(self.widths) - 1)
        return e[e != INVALID]


def level_tables(nodes, had_, widths, leaves=None, discard=False):
    nodes = _c(nodes)
    had_ = _c(had_, np.float32)
    if leaves is None:
        leaves = subtree_leaves(nodes)
    leaves = _c(leaves, np.uint32)
    w = np.asarray(widths, dtype=np.uint32)
    n_ent = n_tab = 0
    nt = 1
    for x in w:
        n_ent += nt * int(x); n_tab += nt; nt *= int(x)
    entry_node = np.empty(n_ent, dtype=np.uint32)
    table_cnt = np.empty(n_tab, dtype=np.uint32)
    _load().oracle_level_tables_ex(nodes.ctypes.data, had_.ctypes.data, leaves.ctypes.data,
                                   w.ctypes.data, len(w), 1 if discard else 0, entry_node.ctypes.data,
                                   table_cnt.ctypes.data)
    return Tables(w, entry_node, table_cnt)


def select_cut(nodes, K, key_bits, lam=0.125):
    """HAD + level tables for a (K, key_bits) request.  Returns (Tables, K_eff, had)."""
    h = had(nodes, lam)
    widths, k_eff = level_widths(K, key_bits)
    return level_tables(nodes, h, widths), k_eff, h


# --------------------------------------------------------------------------- (a2)
def slab_hit(ray, lo, hi):
    ray = _c(ray, np.float32); lo = _c(lo, np.float32); hi = _c(hi, np.float32)
    return bool(_load().oracle_slab_hit(ray.ctypes.data, lo.ctypes.data, hi.ctypes.data))


def encode_hcc(rays, nodes, tables):
    """Hierarchy cut code of every ray; uint64 [n]."""
    rays = _rays(rays); nodes = _c(nodes)
    w = np.asarray(tables.widths, dtype=np.uint32)
    keys = np.empty(rays.shape[0], dtype=np.uint64)
    _load().oracle_encode_hcc(rays.ctypes.data, rays.shape[0], nodes.ctypes.data, w.ctypes.data,
                              len(w), tables.entry_node.ctypes.data, tables.table_cnt.ctypes.data,
                              keys.ctypes.data)
    return keys


def encode_twopoint(rays, scene_lo, scene_hi, key_bits):
    """TwoPoint key; uint64 [n]."""
    rays = _rays(rays)
    lo = _c(scene_lo, np.float32); hi = _c(scene_hi, np.float32)
    keys = np.empty(rays.shape[0], dtype=np.uint64)
    _load().oracle_encode_twopoint(rays.ctypes.data, rays.shape[0], lo.ctypes.data, hi.ctypes.data,
                                   int(key_bits), keys.ctypes.data)
    return keys


def grid_tables(scene_lo, scene_hi, widths):
    """(f4, reading R14) boxes [n_entries, 6] of the regular-grid level tables and
    the per-table counts (all full)."""
    lo = _c(scene_lo, np.float32); hi = _c(scene_hi, np.float32)
    w = np.asarray(widths, dtype=np.uint32)
    n_ent = n_tab = 0
    nt = 1
    for x in w:
        n_ent += nt * int(x); n_tab += nt; nt *= int(x)
    boxes = np.empty((n_ent, 6), dtype=np.float32)
    _load().oracle_grid_tables(lo.ctypes.data, hi.ctypes.data, w.ctypes.data, len(w), boxes.ctypes.data)
    cnt = np.concatenate([np.full(int(np.prod(w[:l], dtype=np.int64)), int(w[l]), dtype=np.uint32) for l in range(len(w))])
    return boxes, cnt


def encode_tables(rays, boxes, widths, table_cnt):
    """The multi-level code over explicit boxes (regular grid, f4); uint64 [n]."""
    rays = _rays(rays); boxes = _c(boxes, np.float32); table_cnt = _c(table_cnt, np.uint32)
    w = np.asarray(widths, dtype=np.uint32)
    keys = np.empty(rays.shape[0], dtype=np.uint64)
    _load().oracle_encode_tables(rays.ctypes.data, rays.shape[0], boxes.ctypes.data, w.ctypes.data, len(w),
                                 table_cnt.ctypes.data, keys.ctypes.data)
    return keys


def encode_ppc(rays, nodes, bits):
    """(f3, reading R13) prefix path code; uint64 [n]."""
    rays = _rays(rays); nodes = _c(nodes)
    keys = np.empty(rays.shape[0], dtype=np.uint64)
    if _load().oracle_encode_ppc(rays.ctypes.data, rays.shape[0], nodes.ctypes.data, int(bits), keys.ctypes.data) != 0:
        raise RuntimeError("oracle_encode_ppc: stack overflow")
    return keys


# --------------------------------------------------------------------------- (a3)
def sort(keys):
    """Stable ascending permutation of ray ids by key; uint32 [n]."""
    keys = _c(keys, np.uint64)
    perm = np.empty(keys.shape[0], dtype=np.uint32)
    if _load().oracle_sort(keys.ctypes.data, keys.shape[0], perm.ctypes.data) != 0:
        raise MemoryError
    return perm


def sort_from_bit(keys, bit_lo):
    """(f1) stable ascending permutation by the keys without their low bit_lo bits."""
    keys = _c(keys, np.uint64)
    perm = np.empty(keys.shape[0], dtype=np.uint32)
    if _load().oracle_sort_from_bit(keys.ctypes.data, keys.shape[0], int(bit_lo), perm.ctypes.data) != 0:
        raise MemoryError
    return perm


# --------------------------------------------------------------------------- (a4)
def tri_hit(ray, tri):
    ray = _c(ray, np.float32); tri = _c(tri, np.float32)
    tuv = np.zeros(3, dtype=np.float32)
    ok = _load().oracle_tri_hit(ray.ctypes.data, tri.ctypes.data, tuv.ctypes.data)
    return bool(ok), tuv


def _hit_arrays(n):
    return (np.empty(n, np.float32), np.empty(n, np.uint32), np.empty(n, np.float32), np.empty(n, np.float32))


def closest_brute(rays, tris):
    rays = _rays(rays); tris = _c(tris, np.float32).reshape(-1, 3, 3)
    t, p, u, v = _hit_arrays(rays.shape[0])
    _load().oracle_closest_brute(rays.ctypes.data, rays.shape[0], tris.ctypes.data, tris.shape[0],
                                 t.ctypes.data, p.ctypes.data, u.ctypes.data, v.ctypes.data)
    return t, p, u, v


def any_brute(rays, tris):
    rays = _rays(rays); tris = _c(tris, np.float32).reshape(-1, 3, 3)
    occ = np.empty(rays.shape[0], np.uint8)
    _load().oracle_any_brute(rays.ctypes.data, rays.shape[0], tris.ctypes.data, tris.shape[0], occ.ctypes.data)
    return occ


def closest_bvh(rays, nodes, prim_idx, tris, stats=False):
    rays = _rays(rays); nodes = _c(nodes); prim_idx = _c(prim_idx, np.uint32)
    tris = _c(tris, np.float32).reshape(-1, 3, 3)
    t, p, u, v = _hit_arrays(rays.shape[0])
    st = np.zeros(2, np.uint64)
    rc = _load().oracle_closest_bvh(rays.ctypes.data, rays.shape[0], nodes.ctypes.data, prim_idx.ctypes.data,
                                    tris.ctypes.data, t.ctypes.data, p.ctypes.data, u.ctypes.data,
                                    v.ctypes.data, st.ctypes.data)
    if rc != 0:
        raise RuntimeError("oracle traversal stack overflow")
    return (t, p, u, v, st) if stats else (t, p, u, v)


def any_bvh(rays, nodes, prim_idx, tris, stats=False):
    rays = _rays(rays); nodes = _c(nodes); prim_idx = _c(prim_idx, np.uint32)
    tris = _c(tris, np.float32).reshape(-1, 3, 3)
    occ = np.empty(rays.shape[0], np.uint8)
    st = np.zeros(2, np.uint64)
    rc = _load().oracle_any_bvh(rays.ctypes.data, rays.shape[0], nodes.ctypes.data, prim_idx.ctypes.data,
                                tris.ctypes.data, occ.ctypes.data, st.ctypes.data)
    if rc != 0:
        raise RuntimeError("oracle traversal stack overflow")
    return (occ, st) if stats else occ
