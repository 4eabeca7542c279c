"""Pins for the oracle's encoders: hierarchy cut code (PAPER.md:146-153 Alg. 1, :192,
:202 Fig. 8), multi-level code (:208-220, Fig. 9 :216), TwoPoint (:92, :241)."""
import os

import numpy as np

import hcc_inputs as hi
import oracle as O

GOLDEN = os.path.join(os.path.dirname(__file__), "golden")


def golden(name):
    out = {}
    for line in open(os.path.join(GOLDEN, name)):
        line = line.split("#")[0].strip()
        if line:
            k, v = line.split()
            out[k] = v
    return out


def ray(o, d, tmin=0.0, tmax=np.inf):
    d = np.asarray(d, np.float64)
    d = d / np.linalg.norm(d)
    return np.array([[o[0], o[1], o[2], tmin, d[0], d[1], d[2], tmax]], np.float32)


def segment(a, b):
    a, b = np.asarray(a, np.float64), np.asarray(b, np.float64)
    return ray(a, b - a, 0.0, np.linalg.norm(b - a))


def boxes_bvh(boxes, counts=None):
    """A BVH whose leaves are the given boxes (left-leaning chain above them).  Only the
    leaves' boxes matter to the encoder; counts set TC and with it the HAD order."""
    k = len(boxes)
    counts = counts or [1] * k
    nodes = []
    # internal chain: node 2i (i < k-1) has children 2i+1 (leaf i) and 2i+2 (rest)
    first = 0
    lo_all = np.min([b[0] for b in boxes], 0)
    hi_all = np.max([b[1] for b in boxes], 0)
    for i in range(k - 1):
        nodes.append((lo_all, hi_all, 2 * i + 1, 0))
        nodes.append((boxes[i][0], boxes[i][1], first, counts[i]))
        first += counts[i]
    nodes.append((boxes[k - 1][0], boxes[k - 1][1], first, counts[k - 1]))
    first += counts[k - 1]
    # fix: the last internal's right child is the last leaf, at index 2(k-1)
    return hi.make_bvh(nodes, np.zeros((first, 3, 3), np.float32))


def manual_tables(widths, entry_lists):
    """Tables from explicit per-level entry arrays (node ids, INVALID padded)."""
    w = np.asarray(widths, np.uint32)
    ent, cnt = [], []
    nt = 1
    for l, wl in enumerate(widths):
        tabs = entry_lists[l]
        assert len(tabs) == nt
        for t in tabs:
            cnt.append(len(t))
            ent.extend(list(t) + [O.INVALID] * (wl - len(t)))
        nt *= wl
    return O.Tables(w, np.asarray(ent, np.uint32), np.asarray(cnt, np.uint32))


# ------------------------------------------------------------------ Fig. 8
def grid_boxes():
    # 4x4 grid in the xy plane, cell (row r, col c) = index 4r + c, unit cells, z in [0,1]
    return [((c, r, 0.0), (c + 1.0, r + 1.0, 1.0)) for r in range(4) for c in range(4)]


def test_fig8_bit_order():
    """sixteen cut nodes; "Ray1 traverses through nodes 0, 1, 5, and 9 ...
    the first, second, sixth, and tenth bits of Ray1's HCC are set to 1".  With node 0 in
    the most significant bit that is 1100 0100 0100 0000."""
    g = golden("fig8_hcc.txt")
    boxes = grid_boxes()
    # TC decreasing with the cell number makes HAD order == cell order (equal areas)
    b = boxes_bvh(boxes, counts=[16 - i for i in range(16)])
    h = O.had(b.nodes)
    c = O.cut(b.nodes, h, 16)
    leaf_of_cell = [2 * i + 1 for i in range(15)] + [30]
    assert list(c) == leaf_of_cell                       # HAD-descending == cell 0..15
    T = O.level_tables(b.nodes, h, [16])
    r1 = segment((0.9, 0.1, 0.5), (1.4, 2.5, 0.5))       # cells 0 -> 1 -> 5 -> 9, ends inside 9
    key = int(O.encode_hcc(r1, b.nodes, T)[0])
    assert key == int(g["ray1"], 2) == 0xC440
    # the same ray unbounded also crosses cell 13
    r1_inf = ray((0.9, 0.1, 0.5), (0.5, 2.4, 0.0))
    assert int(O.encode_hcc(r1_inf, b.nodes, T)[0]) == 0xC444
    # reversing a ray that starts inside the scene changes the code (Ray3/Ray4)
    fwd = ray((2.5, 1.5, 0.5), (1.0, 0.2, 0.0))
    bwd = ray((2.5, 1.5, 0.5), (-1.0, -0.2, 0.0))
    kf, kb = int(O.encode_hcc(fwd, b.nodes, T)[0]), int(O.encode_hcc(bwd, b.nodes, T)[0])
    own = 1 << (15 - 6)                                   # both start in cell 6
    assert kf & own and kb & own and kf != kb and (kf & kb) == own


def test_hcc_short_table_is_right_aligned_and_origin_inside_sets_bit():
    boxes = grid_boxes()[:4]
    b = boxes_bvh(boxes, counts=[4, 3, 2, 1])
    h = O.had(b.nodes)
    T = O.level_tables(b.nodes, h, [4])
    assert T.bits_used == 4
    k = int(O.encode_hcc(ray((2.5, 0.5, 0.5), (0, 0, 1)), b.nodes, T)[0])
    assert k == 0b0010                                    # cell 2 only, key < 2^4
    k = int(O.encode_hcc(ray((-1, 0.5, 0.5), (1, 0, 0)), b.nodes, T)[0])
    assert k == 0b1111
    k = int(O.encode_hcc(ray((-1, 0.5, 0.5), (-1, 0, 0)), b.nodes, T)[0])
    assert k == 0                                         # misses everything


# ------------------------------------------------------------------ Fig. 9
def test_fig9_two_level_layout():
    """16-bit MLHCC = 8 top-level bits above 8 low-level bits; Ray1 is
    printed as 0101110001101100, Ray2 as 0000001100111110.  The figure's geometry is an
    image, so boxes are placed to produce exactly those hit patterns; what is pinned is the
    field layout, the bit order inside a field and the representative rule (:218)."""
    g = golden("fig9_mlhcc.txt")
    top1, low1 = g["ray1"][:8], g["ray1"][8:]
    top2, low2 = g["ray2"][:8], g["ray2"][8:]
    # Ray1 runs along y = 0.5, Ray2 along y = 2.5 (both +x, z = 0.5).  Top boxes: entry j is
    # hit by ray r iff bit j of top_r.  A top box is a union of up to two rows, so give each
    # entry its own x-range and choose which y rows it spans.
    nodes, tris = [], 0

    def add(lo, hi_):
        nonlocal tris
        nodes.append((lo, hi_, tris, 1))
        tris += 1
        return len(nodes) - 1

    def span(b1, b2):
        if b1 == "1" and b2 == "1": return (0.0, 3.0)
        if b1 == "1": return (0.0, 1.0)
        if b2 == "1": return (2.0, 3.0)
        return (4.0, 5.0)                      # off both rays
    top_ids = [add((j, span(top1[j], top2[j])[0], 0.0), (j + 0.9, span(top1[j], top2[j])[1], 1.0))
               for j in range(8)]
    rep1, rep2 = top1.index("1"), top2.index("1")
    assert rep1 == 1 and rep2 == 6
    low_tables = []
    for j in range(8):
        if j == rep1:
            pat = [(low1[i], "0") for i in range(8)]
        elif j == rep2:
            pat = [("0", low2[i]) for i in range(8)]
        else:
            pat = [("1", "1")] * 8            # never consulted: j is not a representative
        low_tables.append([add((j + 0.1 * i, span(*pat[i])[0], 0.0), (j + 0.1 * i + 0.05, span(*pat[i])[1], 1.0))
                           for i in range(8)])
    bvh_nodes = np.zeros(len(nodes), hi.NODE_DTYPE)
    for i, (lo, hi_, f, c) in enumerate(nodes):
        bvh_nodes[i] = (np.float32(lo), np.float32(hi_), f, c)
    T = manual_tables([8, 8], [[top_ids], low_tables])
    r1 = ray((-1.0, 0.5, 0.5), (1, 0, 0))
    r2 = ray((-1.0, 2.5, 0.5), (1, 0, 0))
    k1 = int(O.encode_hcc(r1, bvh_nodes, T)[0])
    k2 = int(O.encode_hcc(r2, bvh_nodes, T)[0])
    assert format(k1, "016b") == g["ray1"] and format(k2, "016b") == g["ray2"]
    # number of set bits = number of boxes crossed: 4 top + 4 low for Ray1
    assert bin(k1 >> 8).count("1") == 4 and bin(k1 & 0xFF).count("1") == 4


# ------------------------------------------------------------------ keys vs independent fp64
def fp64_slab(rays, lo, hi_):
    """Independent statement in float64, by explicit case analysis per axis: the ray's
    parameter interval inside slab a is [enter_a, leave_a] (all t if it runs parallel inside
    the slab, nothing if parallel outside); with [tmin, tmax] as a fourth interval the box is
    hit iff every enter_a <= every leave_b.  Returns (hit, margin): margin is how far the
    closest pair of DIFFERENT intervals is from flipping the decision, relative to the size of
    the numbers (a flat box has enter_a == leave_a on its thin axis: that pair cannot flip)."""
    r = rays.astype(np.float64)
    o, d = r[:, 0:3], r[:, 4:7]
    lo = np.asarray(lo, np.float64); hi_ = np.asarray(hi_, np.float64)
    enter, leave = [r[:, 3]], [r[:, 7]]
    ok = np.ones(len(r), bool)
    for a in range(3):
        par = d[:, a] == 0
        inside = (o[:, a] >= lo[a]) & (o[:, a] <= hi_[a])
        ok &= ~par | inside
        with np.errstate(divide="ignore", invalid="ignore"):
            ta = (lo[a] - o[:, a]) / d[:, a]
            tb = (hi_[a] - o[:, a]) / d[:, a]
        enter.append(np.where(par, -np.inf, np.where(d[:, a] > 0, ta, tb)))
        leave.append(np.where(par, np.inf, np.where(d[:, a] > 0, tb, ta)))
    cross = np.full(len(r), np.inf)
    for a in range(4):
        for b in range(4):
            if a != b:
                with np.errstate(invalid="ignore"):
                    gap = leave[b] - enter[a]
                big = np.maximum(np.where(np.isfinite(enter[a]), np.abs(enter[a]), 0.0),
                                 np.where(np.isfinite(leave[b]), np.abs(leave[b]), 0.0))
                cross = np.minimum(cross, np.where(np.isnan(gap), np.inf, gap) / (1.0 + big))
    return ok & (cross >= 0), np.where(ok, np.abs(cross), np.inf)


def test_keys_match_fp64_slab_tests(tiny, room_small):
    for case, K, B in ((tiny, 64, 32), (room_small, 1024, 32), (room_small, 32, 32), (room_small, 64, 64)):
        n = case.bvh.nodes
        T, _, h = O.select_cut(n, K, B)
        for rays in (case.diffuse, case.shadow):
            keys = O.encode_hcc(rays, n, T)
            assert (keys < (1 << T.bits_used)).all()
            # re-derive every field from scratch, ray by ray, with the fp64 test
            expect = np.zeros(len(rays), np.uint64)
            table = np.zeros(len(rays), np.int64)
            alive = np.ones(len(rays), bool)
            unsure = np.zeros(len(rays), bool)
            for l, w in enumerate(T.widths):
                mask = np.zeros(len(rays), np.uint64)
                rep = np.full(len(rays), -1, np.int64)
                for t in np.unique(table[alive]):
                    sel = alive & (table == t)
                    for j, node in enumerate(T.table(l, int(t))):
                        hit, margin = fp64_slab(rays[sel], n["lo"][node], n["hi"][node])
                        unsure[np.nonzero(sel)[0][margin < 2e-6]] = True
                        idx = np.nonzero(sel)[0][hit]
                        mask[idx] |= np.uint64(1 << (w - 1 - j))
                        first = idx[rep[idx] < 0]
                        rep[first] = j
                expect = (expect << np.uint64(w)) | mask
                alive &= rep >= 0
                table = np.where(alive, table * w + rep, 0)
            good = ~unsure
            assert good.mean() > 0.97
            assert np.array_equal(keys[good], expect[good])


def test_key_structural_invariants(room_small):
    n = room_small.bvh.nodes
    T, _, h = O.select_cut(n, 1024, 32)
    rays = np.concatenate([room_small.diffuse, room_small.shadow])
    keys = O.encode_hcc(rays, n, T)
    w = T.widths
    f1 = keys >> np.uint64(sum(w[1:]))
    # field 1 is the flat mask over the level-1 table
    flat = O.encode_hcc(rays, n, O.level_tables(n, h, [w[0]])) if False else None
    T1 = manual_tables([w[0]], [[list(T.table(0, 0))]])
    assert np.array_equal(f1, O.encode_hcc(rays, n, T1))
    # a lower field can only be non-zero if the field above is (representative rule)
    f2 = (keys >> np.uint64(w[2])) & np.uint64((1 << w[1]) - 1)
    f3 = keys & np.uint64((1 << w[2]) - 1)
    assert not ((f1 == 0) & (f2 != 0)).any() and not ((f2 == 0) & (f3 != 0)).any()
    # rays start inside the room: the level-1 table covers the room, so field 1 is never empty,
    # and a ray whose origin lies inside a cut box sets that box's bit
    assert (f1 != 0).all()
    tab = T.table(0, 0)
    o = rays[:, 0:3]
    for j, node in enumerate(tab):
        inside = ((o >= n["lo"][node]) & (o <= n["hi"][node])).all(1)
        assert ((f1[inside] >> np.uint64(w[0] - 1 - j)) & np.uint64(1)).all()
    # rays that miss the root box get key 0
    out = rays[:64].copy()
    out[:, 0:3] += 5.0
    out[:, 4:7] = np.abs(out[:, 4:7]) + 1e-3
    out[:, 4:7] /= np.linalg.norm(out[:, 4:7], axis=1, keepdims=True)
    assert (O.encode_hcc(out, n, T) == 0).all()


def test_slab_edge_cases():
    lo, hi_ = (0, 0, 0), (1, 1, 1)
    assert O.slab_hit(ray((0.5, 0.5, -1), (0, 0, 1))[0], lo, hi_)           # axis-parallel, inside slabs
    assert not O.slab_hit(ray((1.5, 0.5, -1), (0, 0, 1))[0], lo, hi_)       # axis-parallel, outside a slab
    # exactly in a face plane with d_a = 0: one product is 0*inf = NaN, minNum/maxNum drop it
    # and the other product (-inf or +inf) empties the slab -> defined as a miss (R7)
    assert not O.slab_hit(ray((1.0, 0.5, -1), (0, 0, 1))[0], lo, hi_)
    assert not O.slab_hit(ray((0.0, 0.5, -1), (0, 0, 1))[0], lo, hi_)
    assert O.slab_hit(ray((0.5, 0.5, 0.5), (0, 0, -1))[0], lo, hi_)         # origin inside
    assert not O.slab_hit(ray((0.5, 0.5, 2), (0, 0, 1))[0], lo, hi_)        # box behind the origin
    assert not O.slab_hit(segment((0.5, 0.5, -2), (0.5, 0.5, -1))[0], lo, hi_)   # ends before the box
    assert O.slab_hit(segment((0.5, 0.5, -2), (0.5, 0.5, 0))[0], lo, hi_)        # ends on the face


# ------------------------------------------------------------------ TwoPoint
def test_twopoint_closed_forms():
    lo, hi_ = np.zeros(3, np.float32), np.ones(3, np.float32)
    for B, b in ((16, 2), (24, 4), (32, 5), (48, 8), (64, 10)):
        # origin at the low corner pointing at the high corner, length 0.25*e*|d|: choose d so the
        # estimated end is still the low cell -> all zero
        r = ray((0, 0, 0), (1, 1, 1))
        r[0, 4:7] = 0.0
        assert int(O.encode_twopoint(r, lo, hi_, B)[0]) == 0
        # origin at the high corner (clamped to the last cell), end beyond it: all ones
        r = ray((1, 1, 1), (1, 1, 1))
        assert int(O.encode_twopoint(r, lo, hi_, B)[0]) == (1 << (6 * b)) - 1
        # origin low corner, end point (o + 0.25*d) in the top cell of every axis: 000111 repeated
        r = np.array([[0, 0, 0, 0, 4, 4, 4, np.inf]], np.float32)       # |d| != 1 on purpose: end = (1,1,1)
        pat = int("000111" * b, 2)
        assert int(O.encode_twopoint(r, lo, hi_, B)[0]) == pat
        # only o.x in the upper half: the very first bit
        r = np.array([[0.75, 0, 0, 0, -3, 0, 0, np.inf]], np.float32)   # end x = 0
        assert int(O.encode_twopoint(r, lo, hi_, B)[0]) >> (6 * b - 1) == 1
        # one coordinate in the upper half at a time: o.x o.y o.z t.x t.y t.z from the top bit down (DESIGN.md
        # R10), so y and z cannot be swapped inside either triple.  The end point is o + 0.25 * d (e = 1).
        top6 = lambda ray: int(O.encode_twopoint(np.array([ray], np.float32), lo, hi_, B)[0]) >> (6 * b - 6)
        assert top6([0, 0.75, 0, 0, 0, -3, 0, np.inf]) == 0b010000      # o.y only (end y = 0)
        assert top6([0, 0, 0.75, 0, 0, 0, -3, np.inf]) == 0b001000      # o.z only
        assert top6([0, 0, 0, 0, 3, 0, 0, np.inf]) == 0b000100          # t.x only (end x = 0.75)
        assert top6([0, 0, 0, 0, 0, 3, 0, np.inf]) == 0b000010          # t.y only
        assert top6([0, 0, 0, 0, 0, 0, 3, np.inf]) == 0b000001          # t.z only


def test_twopoint_monotone_and_range(room_small):
    n = room_small.bvh.nodes
    lo, hi_ = n["lo"][0], n["hi"][0]
    k = O.encode_twopoint(room_small.diffuse, lo, hi_, 32)
    assert (k < (1 << 30)).all()
    # moving only o.x upward never lowers the o.x bits (de-interleave and compare)
    r = room_small.diffuse[:512].copy()
    r[:, 4:7] = 0.0
    xs = np.linspace(0, 1, 512, dtype=np.float32)
    r[:, 0] = xs
    kk = O.encode_twopoint(r, lo, hi_, 32)
    ox = np.zeros(512, np.int64)
    for i in range(5):
        ox |= ((kk >> np.uint64(6 * i + 5)) & np.uint64(1)).astype(np.int64) << i
    assert (np.diff(ox) >= 0).all() and ox[0] == 0 and ox[-1] == 31
    assert np.array_equal(ox, np.minimum((xs.astype(np.float64) * 32).astype(np.int64), 31))
