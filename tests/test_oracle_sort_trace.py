"""Pins for the oracle's sort and trace (:247, :62-64; R11, R12)."""
import numpy as np

import hcc_inputs as hi
import oracle as O


# ------------------------------------------------------------------ sort
def test_sort_matches_numpy_stable_argsort():
    rs = np.random.RandomState(5)
    for n, hi_ in ((0, 10), (1, 10), (2, 2), (1000, 7), (4097, 1 << 16), (100003, 1 << 62)):
        keys = rs.randint(0, hi_, size=n, dtype=np.int64).astype(np.uint64)
        perm = O.sort(keys)
        assert perm.dtype == np.uint32
        assert np.array_equal(perm, np.argsort(keys, kind="stable").astype(np.uint32))


def test_sort_properties(room_small):
    n = room_small.bvh.nodes
    T, _, _ = O.select_cut(n, 1024, 32)
    keys = O.encode_hcc(room_small.shadow, n, T)
    perm = O.sort(keys)
    assert np.array_equal(np.sort(perm), np.arange(len(keys)))         # a permutation
    ks = keys[perm]
    assert (ks[:-1] <= ks[1:]).all()                                   # non-decreasing
    same = ks[:-1] == ks[1:]
    assert (perm[:-1][same] < perm[1:][same]).all()                    # equal keys keep id order
    assert np.array_equal(O.sort(np.zeros(100, np.uint64)), np.arange(100))   # all equal -> identity


# ------------------------------------------------------------------ triangle test
def ray(o, d, tmin=0.0, tmax=np.inf):
    return np.array([[o[0], o[1], o[2], tmin, d[0], d[1], d[2], tmax]], np.float32)


def test_tri_hit_closed_forms():
    tri = np.array([[0, 0, 0], [1, 0, 0], [0, 1, 0]], np.float32)      # unit right triangle in z = 0
    ok, tuv = O.tri_hit(ray((0.25, 0.5, 2.0), (0, 0, -1))[0], tri)
    assert ok and tuple(tuv) == (2.0, 0.25, 0.5)                       # t = distance, (u,v) = (x,y)
    ok, _ = O.tri_hit(ray((0.25, 0.5, -2.0), (0, 0, 1))[0], tri)
    assert ok                                                          # no back-face culling
    assert not O.tri_hit(ray((0.6, 0.6, 2.0), (0, 0, -1))[0], tri)[0]  # u + v > 1
    assert not O.tri_hit(ray((-0.1, 0.5, 2.0), (0, 0, -1))[0], tri)[0]
    assert not O.tri_hit(ray((0.25, 0.5, 2.0), (0, 0, 1))[0], tri)[0]  # behind
    assert not O.tri_hit(ray((0.25, 0.5, 2.0), (1, 0, 0))[0], tri)[0]  # parallel: det == 0
    assert not O.tri_hit(ray((0.25, 0.5, 2.0), (0, 0, -1), 0.0, 2.0)[0], tri)[0]   # t < tmax is strict
    assert O.tri_hit(ray((0.25, 0.5, 2.0), (0, 0, -1), 0.0, 2.0001)[0], tri)[0]
    assert not O.tri_hit(ray((0.25, 0.5, 2.0), (0, 0, -1), 2.0, 9.0)[0], tri)[0]   # t > tmin is strict
    # edges and vertices are inside (u >= 0, v >= 0, u + v <= 1 are non-strict)
    assert O.tri_hit(ray((0.0, 0.0, 1.0), (0, 0, -1))[0], tri)[0]
    assert O.tri_hit(ray((0.5, 0.5, 1.0), (0, 0, -1))[0], tri)[0]


def test_aimed_rays_hit_their_triangle(tiny):
    """A ray aimed at a triangle's centroid from distance s along the normal hits at t = s."""
    tris = tiny.bvh.tris[:200].astype(np.float64)
    cen = tris.mean(1)
    nrm = np.cross(tris[:, 1] - tris[:, 0], tris[:, 2] - tris[:, 0])
    nrm /= np.linalg.norm(nrm, axis=1, keepdims=True)
    s = 0.37
    rays = hi.rays.pack_rays(cen + s * nrm, 0.0, -nrm, np.inf)
    for k in range(200):
        ok, tuv = O.tri_hit(rays[k], tiny.bvh.tris[k])
        assert ok and abs(tuv[0] - s) < 1e-5 and abs(tuv[1] - 1 / 3) < 1e-3 and abs(tuv[2] - 1 / 3) < 1e-3


def test_tri_hit_matches_fp64(tiny):
    """Independent fp64 statement (plane intersection + edge functions) on non-grazing cases."""
    rs = np.random.RandomState(3)
    rays = tiny.diffuse[:1500]
    ids = rs.randint(0, tiny.bvh.n_tris, size=len(rays))
    # aim half of them at their triangle so there are plenty of hits
    tri = tiny.bvh.tris[ids].astype(np.float64)
    tgt = (tri * rs.dirichlet((1, 1, 1), size=len(rays))[:, :, None]).sum(1)
    rays = rays.copy()
    d = tgt - rays[:, 0:3]
    d /= np.linalg.norm(d, axis=1, keepdims=True)
    rays[::2, 4:7] = d[::2]
    n_hit = 0
    for k in range(len(rays)):
        r = rays[k].astype(np.float64)
        v0, v1, v2 = tri[k]
        nrm = np.cross(v1 - v0, v2 - v0)
        den = nrm @ r[4:7]
        ok, tuv = O.tri_hit(rays[k], tiny.bvh.tris[ids[k]])
        if abs(den) < 1e-9:
            continue
        t = nrm @ (v0 - r[0:3]) / den
        p = r[0:3] + t * r[4:7]
        area = nrm @ nrm
        b1 = np.cross(p - v0, v2 - v0) @ nrm / area * 1.0      # weight of v1
        b2 = np.cross(v1 - v0, p - v0) @ nrm / area            # weight of v2
        margin = min(b1, b2, 1 - b1 - b2, t)
        if abs(margin) < 1e-4:
            continue
        assert ok == (margin > 0)
        if ok:
            n_hit += 1
            assert abs(tuv[0] - t) <= 1e-5 * max(1.0, t) and abs(tuv[1] - b1) < 1e-4 and abs(tuv[2] - b2) < 1e-4
    assert n_hit > 300


# ------------------------------------------------------------------ traversal == definition
def test_bvh_traversal_equals_brute_force_tiny(tiny):
    """north_star: "traversal hits equal brute-force all-triangle intersection on tiny scenes"."""
    b = tiny.bvh
    prim = tiny.w.primaries(spp=1)
    for rays in (prim, tiny.diffuse):
        t0, p0, u0, v0 = O.closest_brute(rays, b.tris)
        t1, p1, u1, v1 = O.closest_bvh(rays, b.nodes, b.prim_idx, b.tris)
        assert np.array_equal(p0, p1) and np.array_equal(t0, t1)
        assert np.array_equal(u0, u1) and np.array_equal(v0, v1)
        assert ((p0 == O.INVALID) == np.isinf(t0)).all()
    assert (O.closest_brute(prim, b.tris)[1] != O.INVALID).mean() > 0.1
    occ0 = O.any_brute(tiny.shadow, b.tris)
    occ1 = O.any_bvh(tiny.shadow, b.nodes, b.prim_idx, b.tris)
    assert np.array_equal(occ0, occ1) and 0.01 < occ0.mean() < 0.99
    # any-hit is "closest-hit found something" on the same interval
    tc = O.closest_brute(tiny.shadow, b.tris)[1]
    assert np.array_equal(occ0.astype(bool), tc != O.INVALID)


def test_bvh_traversal_equals_brute_force_room_sample(room_small):
    b = room_small.bvh
    d, s = room_small.diffuse[:192], room_small.shadow[:256]
    t0, p0, _, _ = O.closest_brute(d, b.tris)
    t1, p1, _, _ = O.closest_bvh(d, b.nodes, b.prim_idx, b.tris)
    assert np.array_equal(p0, p1) and np.array_equal(t0, t1)
    assert (p0 != O.INVALID).all()                      # closed room: every diffuse ray hits
    assert np.array_equal(O.any_brute(s, b.tris), O.any_bvh(s, b.nodes, b.prim_idx, b.tris))


def test_closest_tie_goes_to_lowest_triangle_id():
    # two coincident triangles: ids 0 and 1 -> id 0 wins whatever the leaf order
    t = np.array([[[0, 0, 0], [1, 0, 0], [0, 1, 0]]] * 2 + [[[0, 0, 5], [1, 0, 5], [0, 1, 5]]], np.float32)
    for order in ([0, 1, 2], [1, 0, 2], [2, 1, 0]):
        b = hi.make_bvh([((0, 0, 0), (1, 1, 5), 0, 3)], t, prim_idx=order)
        r = ray((0.2, 0.2, -1), (0, 0, 1))
        tt, pp, _, _ = O.closest_bvh(r, b.nodes, b.prim_idx, b.tris)
        assert pp[0] == 0 and tt[0] == 1.0
        assert O.closest_brute(r, t)[1][0] == 0
