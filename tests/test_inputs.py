"""The generated inputs (scenes, host BVH, rays): structure, counts, determinism."""
import numpy as np

import hcc_inputs as hi
from conftest import ancestors_of


def check_bvh(bvh, max_leaf=4):
    nodes = bvh.nodes
    n = nodes.shape[0]
    internal = nodes["count"] == 0
    left = nodes["left_or_first"][internal].astype(np.int64)
    idx = np.nonzero(internal)[0]
    assert (left > idx).all() and (left + 1 < n).all()                 # parent index < child index
    # every node except the root is the child of exactly one node, siblings adjacent
    kids = np.sort(np.concatenate([left, left + 1]))
    assert np.array_equal(kids, np.arange(1, n))
    leaves = ~internal
    assert (nodes["count"][leaves] <= max_leaf).all() and (nodes["count"][leaves] >= 1).all()
    # leaf ranges tile prim_idx exactly once
    first = nodes["left_or_first"][leaves].astype(np.int64)
    cnt = nodes["count"][leaves].astype(np.int64)
    cover = np.zeros(bvh.n_tris, dtype=np.int64)
    for f, c in zip(first, cnt):
        cover[f:f + c] += 1
    assert (cover == 1).all()
    assert np.array_equal(np.sort(bvh.prim_idx), np.arange(bvh.n_tris))
    # leaf boxes are the exact bounds of their triangles; internal boxes the union of the children
    for i in np.nonzero(leaves)[0][:2000]:
        t = bvh.tris[bvh.prim_idx[nodes["left_or_first"][i]:nodes["left_or_first"][i] + nodes["count"][i]]]
        assert np.array_equal(nodes["lo"][i], t.reshape(-1, 3).min(0))
        assert np.array_equal(nodes["hi"][i], t.reshape(-1, 3).max(0))
    l = nodes["left_or_first"][idx]
    assert np.array_equal(nodes["lo"][idx], np.minimum(nodes["lo"][l], nodes["lo"][l + 1]))
    assert np.array_equal(nodes["hi"][idx], np.maximum(nodes["hi"][l], nodes["hi"][l + 1]))


def test_scene_counts():
    assert hi.make_scene("tiny").shape == (1024, 3, 3)
    assert hi.make_scene("room").shape == (64012, 3, 3)          # 12 + 200*320
    assert hi.scenes.icosphere(2).shape[0] == 320
    assert hi.scenes.icosphere(4).shape[0] == 5120
    s = hi.make_scene("fig1", scale=0.01)
    assert s.shape[0] == 12 + 2 * 5120 + 65 * 12


def test_scene_inside_room_and_deterministic():
    a = hi.make_scene("room")
    b = hi.make_scene("room")
    assert a.dtype == np.float32 and np.array_equal(a, b)
    assert a.min() >= 0.0 and a.max() <= 1.0
    e = np.linalg.norm(hi.make_scene("tiny")[:, 1] - hi.make_scene("tiny")[:, 0], axis=1)
    assert e.min() > 0.0099 and e.max() < 0.0501


def test_bvh_structure_tiny(tiny):
    check_bvh(tiny.bvh)
    assert tiny.bvh.max_depth < 64


def test_bvh_structure_room(room_small):
    check_bvh(room_small.bvh)
    parent = ancestors_of(room_small.bvh.nodes)
    assert parent[0] == -1 and (parent[1:] >= 0).all()


def test_bvh_degenerate_coincident_centres():
    t = np.tile(np.array([[[0, 0, 0], [1, 0, 0], [0, 1, 0]]], np.float32), (9, 1, 1))
    b = hi.build_bvh(t)
    check_bvh(b)
    assert b.n_leaves >= 3


def test_ray_batches(tiny, room_small):
    for case, nd in ((tiny, 4096), (room_small, 64 * 64)):
        d, s = case.diffuse, case.shadow
        assert d.shape == (nd, 8) and s.shape == (2 * nd, 8) and d.dtype == np.float32
        for r in (d, s):
            assert np.abs(np.linalg.norm(r[:, 4:7], axis=1) - 1.0).max() < 1e-6
            assert (r[:, 3] == 0).all()
        assert np.isinf(d[:, 7]).all() and np.isfinite(s[:, 7]).all() and (s[:, 7] > 0).all()
        # both shadow rays of a hit share the diffuse ray's origin
        assert np.array_equal(s[0::2, 0:3], d[:, 0:3]) and np.array_equal(s[1::2, 0:3], d[:, 0:3])


def test_rng_uniform():
    u = hi.rng.u01(7, 1, np.arange(200000), 0)
    assert 0.0 <= u.min() and u.max() < 1.0
    assert abs(u.mean() - 0.5) < 0.005 and abs(u.var() - 1 / 12) < 0.002
    assert not np.array_equal(u, hi.rng.u01(7, 1, np.arange(200000), 1))
