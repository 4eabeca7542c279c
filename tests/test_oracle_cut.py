"""Pins for the oracle's HAD (Eq. 1) and cut search (Alg. 2 :171-183,
Alg. 3 :222-231, ordering :192).  Nothing here calls the CUDA path."""
import os

import numpy as np
import pytest

import hcc_inputs as hi
import oracle as O
from conftest import ancestors_of

GOLDEN = os.path.join(os.path.dirname(__file__), "golden")


def box_node(lo, hi, lf, c):
    return (lo, hi, lf, c)


def dummy_tris(n):
    return np.zeros((n, 3, 3), np.float32)


def perfect_tree(depth):
    """Heap-numbered perfect binary tree; a node at depth d covers an x-interval of
    length 2^-d of the unit cube; every leaf holds one triangle."""
    nodes = []
    n_leaf = 0
    for i in range(2 ** (depth + 1) - 1):
        d = int(np.floor(np.log2(i + 1)))
        j = i + 1 - 2 ** d
        lo = (j / 2 ** d, 0.0, 0.0)
        hi_ = ((j + 1) / 2 ** d, 1.0, 1.0)
        if d == depth:
            nodes.append(box_node(lo, hi_, n_leaf, 1)); n_leaf += 1
        else:
            nodes.append(box_node(lo, hi_, 2 * i + 1, 0))
    return hi.make_bvh(nodes, dummy_tris(n_leaf))


# ------------------------------------------------------------------ HAD
def test_had_two_leaf_closed_form():
    # Eq. 1 by hand: leaves TC*SA, root HAD_l + HAD_r + 0.125*SA
    b = hi.make_bvh([box_node((0, 0, 0), (2, 1, 1), 1, 0),
                     box_node((0, 0, 0), (1, 1, 1), 0, 3),        # SA = 6,  TC = 3 -> 18
                     box_node((1, 0, 0), (2, 1, 0.5), 3, 2)],     # SA = 2(1+.5+.5)=4, TC = 2 -> 8
                    dummy_tris(5))
    h = O.had(b.nodes, 0.125)
    assert h[1] == 18.0 and h[2] == 8.0
    assert h[0] == 18.0 + 8.0 + 0.125 * 10.0                      # SA(root) = 2(2+1+2) = 10
    h1 = O.had(b.nodes, 1.0)
    assert h1[0] == 36.0


def test_had_lambda_zero_is_sum_of_leaf_terms(tiny):
    n = tiny.bvh.nodes
    h = O.had(n, 0.0)
    leaf = n["count"] > 0
    assert abs(float(h[0]) - float(h[leaf].astype(np.float64).sum())) <= 1e-4 * float(h[0])


def test_had_matches_fp64_and_is_monotone(room_small):
    n = room_small.bvh.nodes
    h = O.had(n)
    ext = (n["hi"].astype(np.float64) - n["lo"].astype(np.float64))
    sa = 2.0 * (ext[:, 0] * ext[:, 1] + ext[:, 1] * ext[:, 2] + ext[:, 2] * ext[:, 0])
    ref = np.zeros(len(n))
    for k in range(len(n) - 1, -1, -1):
        if n["count"][k] > 0:
            ref[k] = n["count"][k] * sa[k]
        else:
            l = n["left_or_first"][k]
            ref[k] = ref[l] + ref[l + 1] + 0.125 * sa[k]
    assert np.allclose(h, ref, rtol=2e-5, atol=0)
    parent = ancestors_of(n)
    assert (h[parent[1:]] >= h[1:]).all()            # parent >= child: all terms are >= 0


# ------------------------------------------------------------------ Alg. 2
def cut_invariants(nodes, cut, K):
    parent = ancestors_of(nodes)
    cs = set(int(c) for c in cut)
    assert len(cs) == len(cut)
    n_leaves = int((nodes["count"] > 0).sum())
    assert len(cut) == min(K, n_leaves)
    # every leaf has exactly one ancestor-or-self in the cut  (antichain + cover)
    for leaf in np.nonzero(nodes["count"] > 0)[0]:
        k, hits = int(leaf), 0
        while k >= 0:
            hits += k in cs
            k = int(parent[k])
        assert hits == 1


def closed_form_cut(nodes, had, K):
    """Frontier of the K-1 highest-HAD internal nodes (HAD desc, index asc): the
    data-parallel restatement of Alg. 2; valid because HAD is monotone
    and leaf pops never advance the loop."""
    internal = np.nonzero(nodes["count"] == 0)[0]
    order = internal[np.lexsort((internal, -had[internal].astype(np.float64)))]
    S = order[:max(K - 1, 0)]
    if len(S) == 0:
        return {0}
    inS = np.zeros(len(nodes), bool)
    inS[S] = True
    kids = np.concatenate([nodes["left_or_first"][S], nodes["left_or_first"][S] + 1])
    return set(int(k) for k in kids if not inS[k])


@pytest.mark.parametrize("K", [1, 2, 3, 7, 16, 32, 64, 100, 333])
def test_alg2_invariants_and_closed_form_tiny(tiny, K):
    n = tiny.bvh.nodes
    h = O.had(n)
    c = O.cut(n, h, K)
    cut_invariants(n, c, K)
    assert set(int(x) for x in c) == closed_form_cut(n, h, K)
    # HAD descending, ties -> lower index
    hv = h[c]
    assert (hv[:-1] >= hv[1:]).all()
    assert all(c[i] < c[i + 1] for i in range(len(c) - 1) if hv[i] == hv[i + 1])


@pytest.mark.parametrize("K", [256, 1024, 4096, 20000])
def test_alg2_closed_form_room(room_small, K):
    n = room_small.bvh.nodes
    h = O.had(n)
    c = O.cut(n, h, K)
    assert len(c) == K
    assert set(int(x) for x in c) == closed_form_cut(n, h, K)


def test_alg2_special_cases(tiny):
    n = tiny.bvh.nodes
    h = O.had(n)
    assert list(O.cut(n, h, 1)) == [0]                                  # K = 1 -> root
    n_leaves = tiny.bvh.n_leaves
    for K in (n_leaves, n_leaves + 5, 10 * n_leaves):                   # K >= #leaves -> all leaves
        c = O.cut(n, h, K)
        assert set(int(x) for x in c) == set(np.nonzero(n["count"] > 0)[0].tolist())


def test_alg2_breadth_first_on_perfect_tree():
    # PAPER.md:169 "The search goes in breadth-first order", :517
    b = perfect_tree(6)
    h = O.had(b.nodes)
    for d in range(0, 7):
        c = O.cut(b.nodes, h, 2 ** d)
        assert sorted(int(x) for x in c) == list(range(2 ** d - 1, 2 ** (d + 1) - 1))


def test_alg2_leaf_rule_fig7():
    """PAPER.md:157/:169 Fig. 7 narrative: an unbalanced BVH; a leaf is popped during the
    search, is kept as a cut node and is no longer searched; seven cut nodes are found."""
    # 0 root -> 1 (LEAF), 2;  2 -> 3,4;  3 -> 5,6;  4 -> 7,8;  5..8 -> two leaves each (9..16)
    nodes = [box_node((0, 0, 0), (1, 1, 1), 1, 0), box_node((0, 0, 0), (1, 1, 1), 0, 4),
             box_node((0, 0, 0), (1, 1, 1), 3, 0), box_node((0, 0, 0), (1, 1, 1), 5, 0),
             box_node((0, 0, 0), (1, 1, 1), 7, 0), box_node((0, 0, 0), (1, 1, 1), 9, 0),
             box_node((0, 0, 0), (1, 1, 1), 11, 0), box_node((0, 0, 0), (1, 1, 1), 13, 0),
             box_node((0, 0, 0), (1, 1, 1), 15, 0)]
    for k in range(8):
        nodes.append(box_node((0, 0, 0), (1, 1, 1), 4 + k, 1))
    b = hi.make_bvh(nodes, dummy_tris(12))
    # priorities chosen by hand (the search only reads this array): the leaf 1 outranks node 2
    had = np.array([100, 60, 50, 30, 20, 12, 11, 9, 8, 6, 5, 4, 3, 2, 2, 1, 1], np.float32)
    c = O.cut(b.nodes, had, 7)
    # by hand: pop 0 -> {1,2}; pop 1 (leaf: retired, Max 7->6); pop 2 -> {3,4}; pop 3 -> {4,5,6};
    # pop 4 -> {5,6,7,8}; pop 5 -> {6,7,8,9,10}; pop 6 -> {7,8,9,10,11,12}: 6 in queue = Max, stop.
    assert list(c) == [1, 7, 8, 9, 10, 11, 12]
    cut_invariants(b.nodes, c, 7)
    # K larger than the number of leaves (9): the queue drains, every leaf is returned
    assert sorted(O.cut(b.nodes, had, 50).tolist()) == [1, 9, 10, 11, 12, 13, 14, 15, 16]
    # "large enough" counts LEAVES below a node, not triangles (the subtree must be able to
    # fill the next level's table with cut nodes): leaf 1 holds four triangles and still counts once
    assert b.nodes["count"][1] == 4
    assert O.subtree_leaves(b.nodes).tolist() == [9, 1, 8, 4, 4, 2, 2, 2, 2, 1, 1, 1, 1, 1, 1, 1, 1]


def test_alg2_tie_break_lower_index():
    b = perfect_tree(2)                     # 7 nodes, all priorities equal
    had = np.ones(7, np.float32)
    assert list(O.cut(b.nodes, had, 2)) == [1, 2]
    assert list(O.cut(b.nodes, had, 3)) == [2, 3, 4]      # node 1 (lower index) popped before 2


# ------------------------------------------------------------------ Alg. 3 / level tables
def test_level_width_rule_golden():
    """Reading R-ML; the table is tests/golden/level_widths.txt."""
    for line in open(os.path.join(GOLDEN, "level_widths.txt")):
        line = line.split("#")[0].strip()
        if not line:
            continue
        K, B, widths, keff = line.split()
        w, ke = O.level_widths(int(K), int(B))
        assert w == [int(x) for x in widths.split("x")], line
        assert ke == int(keff), line
        assert sum(w) <= int(B)
        if len(w) > 1:
            assert int(np.prod(w)) == ke


@pytest.mark.parametrize("K,B", [(64, 32), (1024, 32), (4096, 64), (256, 16), (64, 64), (20, 32)])
def test_level_tables_structure(room_small, K, B):
    n = room_small.bvh.nodes
    T, keff, h = O.select_cut(n, K, B)
    parent = ancestors_of(n)
    m = len(T.widths)
    leaves = O.subtree_leaves(n)
    # level 0 with need=2 is Alg. 2 itself; with need = w[1] it is Alg. 3 in reading R4
    need0 = T.widths[1] if m > 1 else 2
    assert list(T.table(0, 0)) == list(O.cut(n, h, T.widths[0], need=need0))
    for l in range(m):
        ent = T.level_entries(l)
        valid = ent[ent != O.INVALID]
        cut_invariants(n, valid, len(valid))                 # every level is a cut
        assert len(valid) <= int(np.prod(T.widths[:l + 1]))
        w = T.widths[l]
        for t in range(T.n_tables[l]):
            tab = T.table(l, t)
            hv = h[tab]
            assert (hv[:-1] >= hv[1:]).all()                 # PAPER.md:218 sorted by HAD
            if l > 0:
                par = T.level_entries(l - 1)[t]
                if par == O.INVALID:
                    assert len(tab) == 0
                    continue
                assert len(tab) >= 1
                for e in tab:                               # nested refinement of the parent entry
                    k = int(e)
                    while k != int(par) and k >= 0:
                        k = int(parent[k])
                    assert k == int(par)
                # a parent that is a leaf / too small for the next level is kept whole
                if n["count"][par] > 0 or leaves[par] < w:
                    pass
                if n["count"][par] > 0:
                    assert list(tab) == [par]
    assert len(T.finest_cut()) <= keff
    if m == 1:
        assert list(T.table(0, 0)) == list(O.cut(n, h, K))   # plain HCC: Alg. 2 verbatim


def test_alg3_need_keeps_small_subtrees_whole():
    b = perfect_tree(3)                    # 8 leaves
    h = O.had(b.nodes)
    # need = 8: only the root (8 leaves) is expandable -> {1, 2}, whatever K asks for
    assert sorted(O.cut(b.nodes, h, 4, need=8).tolist()) == [1, 2]
    # need = 4: root and depth-1 nodes expandable -> depth 2
    assert sorted(O.cut(b.nodes, h, 4, need=4).tolist()) == [3, 4, 5, 6]
    assert sorted(O.cut(b.nodes, h, 8, need=4).tolist()) == [3, 4, 5, 6]
