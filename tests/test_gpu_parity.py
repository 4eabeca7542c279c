"""Parity of the CUDA path (through the C ABI, via the thin binding) against the oracle, on
the same seeded inputs.  Bars (BASELINE.json north_star): cut node sets, keys and the
stable-sorted permutation bit-exact; hit prim ids identical wherever the two nearest
candidate t differ by more than 1e-5 relative; hit t within 1e-5 relative; any-hit bits
identical."""
import numpy as np
import pytest

pytestmark = pytest.mark.gpu

torch = pytest.importorskip("torch")

REL_T = 1e-5


@pytest.fixture(scope="module")
def hcc():
    if not torch.cuda.is_available():
        pytest.skip("no CUDA device")
    import paper_2305_16652_b200 as h
    return h


@pytest.fixture(scope="module")
def dev_cases(hcc, tiny, room_small, room_mid):
    out = {}
    for name, case in (("tiny", tiny), ("room_small", room_small), ("room_mid", room_mid)):
        b = case.bvh
        out[name] = dict(case=case, bvh=hcc.Bvh(b.nodes, b.tris, b.prim_idx),
                         diffuse=torch.from_numpy(case.diffuse).cuda(),
                         shadow=torch.from_numpy(case.shadow).cuda())
    return out


def _u32(t):
    return t.detach().cpu().numpy().view(np.uint32)


# ------------------------------------------------------------------------------- (a1)
@pytest.mark.parametrize("name", ["tiny", "room_small"])
@pytest.mark.parametrize("lam", [0.125, 0.3, 1.0])
def test_density_bit_exact(hcc, dev_cases, name, lam):
    import oracle
    d = dev_cases[name]
    got = hcc.density(d["bvh"], lam).cpu().numpy()
    want = oracle.had(d["case"].bvh.nodes, lam)
    assert np.array_equal(got.view(np.uint32), want.view(np.uint32))


def test_bvh_info(hcc, dev_cases):
    for d in dev_cases.values():
        b = d["case"].bvh
        assert d["bvh"].n_nodes == b.n_nodes and d["bvh"].n_tris == b.n_tris
        assert d["bvh"].n_leaves == b.n_leaves and d["bvh"].max_depth == b.max_depth
        assert np.array_equal(d["bvh"].scene_lo, b.nodes["lo"][0]) and np.array_equal(d["bvh"].scene_hi, b.nodes["hi"][0])


CUT_REQUESTS = [(1, 32), (2, 16), (16, 16), (32, 32), (64, 64), (64, 32), (64, 16), (256, 32), (256, 16),
                (1024, 32), (1024, 64), (4096, 64), (4096, 24), (16384, 64), (65536, 64), (65536, 32),
                (48, 48), (100, 32), (1000, 48)]


@pytest.mark.parametrize("name", ["tiny", "room_small"])
@pytest.mark.parametrize("K,bits", CUT_REQUESTS)
def test_select_cut_tables_bit_exact(hcc, dev_cases, name, K, bits):
    import oracle
    d = dev_cases[name]
    nodes = d["case"].bvh.nodes
    had = hcc.density(d["bvh"])
    cut = hcc.select_cut(d["bvh"], had, K, bits)
    info = cut.info()
    tables, k_eff, _ = oracle.select_cut(nodes, K, bits)
    assert info["widths"] == tables.widths and info["K_eff"] == k_eff
    assert info["bits_used"] == tables.bits_used and info["container_bits"] == (32 if bits <= 32 else 64)
    ent, cnt = cut.read()
    assert np.array_equal(cnt, tables.table_cnt)
    assert np.array_equal(ent, tables.entry_node)
    cut.close()


@pytest.mark.parametrize("widths,bits", [([8, 8], 16), ([16, 16], 32), ([32, 32], 64), ([4, 4, 4, 4], 16),
                                         ([64], 64), ([3, 5, 7], 16), ([16, 8, 8], 32), ([1, 1, 2], 16)])
def test_select_cut_levels_bit_exact(hcc, dev_cases, widths, bits):
    import oracle
    d = dev_cases["room_small"]
    nodes = d["case"].bvh.nodes
    had = hcc.density(d["bvh"])
    cut = hcc.select_cut_levels(d["bvh"], had, widths, bits)
    tables = oracle.level_tables(nodes, oracle.had(nodes), widths)
    ent, cnt = cut.read()
    assert np.array_equal(cnt, tables.table_cnt) and np.array_equal(ent, tables.entry_node)


@pytest.mark.parametrize("name", ["tiny", "room_small"])
def test_select_cut_flat_any_K(hcc, dev_cases, name):
    import oracle
    d = dev_cases[name]
    nodes = d["case"].bvh.nodes
    had_o = oracle.had(nodes)
    had = hcc.density(d["bvh"])
    n_leaves = d["case"].bvh.n_leaves
    for K in [1, 2, 3, 7, 64, 65, 1000, 4096, 5000, n_leaves - 1, n_leaves, n_leaves + 5]:
        out, cnt = hcc.select_cut_flat(d["bvh"], had, K)
        c = int(cnt.cpu()[0])
        want = oracle.cut(nodes, had_o, K)
        assert c == want.shape[0] == min(K, n_leaves)
        assert np.array_equal(_u32(out)[:c], want), K


# ------------------------------------------------------------------------------- (a2)
# (4096, 24) and (65536, 32) are six and eight levels of 4 (the hierarchies bench.py --studies sweeps); (16384, 48)
# and (65536, 64) have level tables past the 160 KB that fit shared memory (the global-memory branch of the encoder)
# (256, 32) and (1024, 64) are the paper's own two compressed encoders, MLHCC32 = 16 x 16 and MLHCC64 = 32 x 32
# (tests/golden/level_widths.txt)
ENC_REQUESTS = [(64, 32), (32, 32), (64, 64), (1024, 32), (4096, 64), (16384, 64), (256, 16), (48, 48), (1000, 48),
                (4096, 24), (65536, 32), (16384, 48), (65536, 64), (256, 32), (1024, 64)]


@pytest.mark.parametrize("name", ["tiny", "room_mid"])
@pytest.mark.parametrize("K,bits", ENC_REQUESTS)
def test_encode_keys_bit_exact(hcc, dev_cases, name, K, bits):
    import oracle
    d = dev_cases[name]
    nodes = d["case"].bvh.nodes
    tables, _, _ = oracle.select_cut(nodes, K, bits)
    cut = hcc.select_cut(d["bvh"], hcc.density(d["bvh"]), K, bits)
    for batch in ("diffuse", "shadow"):
        got = hcc.keys_to_numpy(hcc.encode(d[batch], cut))
        want = oracle.encode_hcc(getattr(d["case"], batch), nodes, tables)
        assert np.array_equal(got, want), (batch, int((got != want).sum()))
        assert int(got.max()) < (1 << tables.bits_used)


def test_encode_degenerate_rays(hcc, dev_cases):
    """Axis-parallel directions (0 components), origins on box planes, rays missing the scene."""
    import oracle
    d = dev_cases["room_small"]
    nodes = d["case"].bvh.nodes
    rng = np.random.default_rng(5)
    n = 5000
    rays = np.zeros((n, 8), np.float32)
    rays[:, 0:3] = rng.uniform(-0.5, 1.5, (n, 3))
    dirs = rng.normal(size=(n, 3))
    dirs[rng.uniform(size=(n, 3)) < 0.4] = 0.0
    dirs[np.abs(dirs).sum(1) == 0, 0] = 1.0
    dirs[rng.uniform(size=(n, 3)) < 0.1] *= -0.0
    rays[:, 4:7] = dirs / np.linalg.norm(dirs, axis=1, keepdims=True)
    rays[:, 7] = np.where(rng.uniform(size=n) < 0.5, np.inf, rng.uniform(0.01, 2.0, n))
    # origins snapped onto cut-box planes
    tables, _, _ = oracle.select_cut(nodes, 1024, 32)
    boxes = nodes[tables.level_entries(0)[: tables.table_cnt[0]]]
    for i in range(0, n, 7):
        b = boxes[i % boxes.shape[0]]
        a = i % 3
        rays[i, a] = b["lo"][a] if (i // 3) % 2 else b["hi"][a]
    cut = hcc.select_cut(d["bvh"], hcc.density(d["bvh"]), 1024, 32)
    got = hcc.keys_to_numpy(hcc.encode(torch.from_numpy(rays).cuda(), cut))
    want = oracle.encode_hcc(rays, nodes, tables)
    assert np.array_equal(got, want)


@pytest.mark.parametrize("bits", [16, 24, 32, 48, 64])
def test_twopoint_keys_bit_exact(hcc, dev_cases, bits):
    import oracle
    for name in ("tiny", "room_mid"):
        d = dev_cases[name]
        lo, hi = d["bvh"].scene_lo, d["bvh"].scene_hi
        for batch in ("diffuse", "shadow"):
            got = hcc.keys_to_numpy(hcc.encode_twopoint(d[batch], lo, hi, bits))
            want = oracle.encode_twopoint(getattr(d["case"], batch), lo, hi, bits)
            assert np.array_equal(got, want)


# ------------------------------------------------------------------------------- (a3)
@pytest.mark.parametrize("cb", [32, 64])
@pytest.mark.parametrize("n", [1, 2, 31, 33, 4095, 4096, 4097, 8192 + 5, 100003, 1 << 20])
def test_sort_random_keys(hcc, cb, n):
    import oracle
    rng = np.random.default_rng(n * 3 + cb)
    for bits_used in ([5, 8, 16, 20, 32] if cb == 32 else [9, 32, 40, 48, 64]):
        if n > 200000 and bits_used not in (32, 48):
            continue
        hi = (1 << bits_used) - 1
        keys = rng.integers(0, hi, size=n, dtype=np.uint64, endpoint=True)
        if bits_used >= 16:         # long runs of equal keys exercise stability
            keys[rng.uniform(size=n) < 0.3] = keys[0]
        dt = np.uint32 if cb == 32 else np.uint64
        kd = torch.from_numpy(keys.astype(dt).view(np.int32 if cb == 32 else np.int64)).cuda()
        perm = _u32(hcc.sort(kd, bits_used))
        assert np.array_equal(perm, oracle.sort(keys)), (n, cb, bits_used)


def test_sort_zero_bits_and_empty(hcc):
    kd = torch.zeros(1000, dtype=torch.int32, device="cuda")
    assert np.array_equal(_u32(hcc.sort(kd, 0)), np.arange(1000, dtype=np.uint32))
    e = torch.zeros(0, dtype=torch.int32, device="cuda")
    assert hcc.sort(e, 32).shape[0] == 0


@pytest.mark.parametrize("name,K,bits", [("tiny", 64, 32), ("room_mid", 1024, 32), ("room_mid", 4096, 64)])
def test_sort_of_encoded_keys(hcc, dev_cases, name, K, bits):
    import oracle
    d = dev_cases[name]
    cut = hcc.select_cut(d["bvh"], hcc.density(d["bvh"]), K, bits)
    for batch in ("diffuse", "shadow"):
        keys = hcc.encode(d[batch], cut)
        k_host = hcc.keys_to_numpy(keys)
        perm = _u32(hcc.sort(keys, cut.info()["bits_used"]))
        assert np.array_equal(perm, oracle.sort(k_host))


# ------------------------------------------------------------------------------- (a4)
def _second_nearest_gap_ok(case, rays, idx, t_first):
    """For the rays `idx` where prim ids differ: True where the two nearest candidate t are
    within REL_T relative of each other (then either prim is a correct answer)."""
    import oracle
    ok = np.zeros(idx.shape[0], dtype=bool)
    tris = case.bvh.tris.reshape(-1, 9)
    for j, i in enumerate(idx):
        ts = []
        for k in range(tris.shape[0]):
            hit, tuv = oracle.tri_hit(rays[i], tris[k])
            if hit:
                ts.append(float(tuv[0]))
        ts.sort()
        ok[j] = len(ts) >= 2 and (ts[1] - ts[0]) <= REL_T * abs(ts[0])
    return ok


def check_closest(case, rays, got, want):
    gt, gp, gu, gv = got
    wt, wp, wu, wv = want
    assert np.array_equal(np.isinf(gt), np.isinf(wt)), "hit / miss sets differ"
    hit = ~np.isinf(wt)
    assert np.all(gp[~hit] == 0xFFFFFFFF)
    rel = np.abs(gt[hit] - wt[hit]) / np.abs(wt[hit])
    assert rel.size == 0 or rel.max() <= REL_T, rel.max()
    diff = np.nonzero(gp != wp)[0]
    assert diff.shape[0] <= 64, f"{diff.shape[0]} prim ids differ"
    if diff.shape[0]:
        assert _second_nearest_gap_ok(case, rays, diff, wt).all()
    same = hit & (gp == wp)
    assert np.allclose(gu[same], wu[same], rtol=0, atol=1e-4) and np.allclose(gv[same], wv[same], rtol=0, atol=1e-4)


@pytest.mark.parametrize("name", ["tiny", "room_small", "room_mid"])
def test_trace_closest_vs_oracle(hcc, dev_cases, name):
    import oracle
    d = dev_cases[name]
    b = d["case"].bvh
    want = oracle.closest_bvh(d["case"].diffuse, b.nodes, b.prim_idx, b.tris)
    got = hcc.hits_to_numpy(hcc.trace(d["bvh"], d["diffuse"], None, hcc.TRACE_CLOSEST))
    check_closest(d["case"], d["case"].diffuse, got, want)


@pytest.mark.parametrize("name", ["tiny", "room_small", "room_mid"])
def test_trace_any_vs_oracle(hcc, dev_cases, name):
    import oracle
    d = dev_cases[name]
    b = d["case"].bvh
    want = oracle.any_bvh(d["case"].shadow, b.nodes, b.prim_idx, b.tris)
    got = hcc.trace(d["bvh"], d["shadow"], None, hcc.TRACE_ANY).cpu().numpy()
    assert np.array_equal(got, want)
    assert 0 < int(want.sum()) < want.shape[0]


def test_trace_tiny_vs_brute_force(hcc, dev_cases):
    """Config 1: the definition itself (all-triangle intersection)."""
    import oracle
    d = dev_cases["tiny"]
    case = d["case"]
    want = oracle.closest_brute(case.diffuse, case.bvh.tris)
    got = hcc.hits_to_numpy(hcc.trace(d["bvh"], d["diffuse"], None, hcc.TRACE_CLOSEST))
    check_closest(case, case.diffuse, got, want)
    occ = hcc.trace(d["bvh"], d["shadow"], None, hcc.TRACE_ANY).cpu().numpy()
    assert np.array_equal(occ, oracle.any_brute(case.shadow, case.bvh.tris))


def test_trace_primary_rays_with_misses(hcc, dev_cases):
    import oracle
    d = dev_cases["tiny"]
    case = d["case"]
    prim = case.w.primaries()
    want = oracle.closest_bvh(prim, case.bvh.nodes, case.bvh.prim_idx, case.bvh.tris)
    got = hcc.hits_to_numpy(hcc.trace(d["bvh"], torch.from_numpy(prim).cuda(), None, hcc.TRACE_CLOSEST))
    assert np.isinf(want[0]).any() and (~np.isinf(want[0])).any()
    check_closest(case, prim, got, want)


@pytest.mark.parametrize("name,K,bits", [("tiny", 64, 32), ("room_mid", 1024, 32)])
def test_trace_through_perm_writes_by_ray_id(hcc, dev_cases, name, K, bits):
    """Thread j traces ray perm[j]; results land at the ray's own index, so the
    reordered results are bit-identical to the NoSort ones."""
    d = dev_cases[name]
    cut = hcc.select_cut(d["bvh"], hcc.density(d["bvh"]), K, bits)
    for batch, mode in (("diffuse", hcc.TRACE_CLOSEST), ("shadow", hcc.TRACE_ANY)):
        perm = hcc.sort(hcc.encode(d[batch], cut), cut.info()["bits_used"])
        a = hcc.trace(d["bvh"], d[batch], None, mode)
        b = hcc.trace(d["bvh"], d[batch], perm, mode)
        assert torch.equal(a.view(torch.uint8), b.view(torch.uint8))


def test_trace_stats_and_anc(hcc, dev_cases):
    import oracle
    d = dev_cases["room_small"]
    b = d["case"].bvh
    st = hcc.trace_stats(d["bvh"], d["diffuse"], None, hcc.TRACE_CLOSEST)
    assert st["rays"] == d["diffuse"].shape[0] and st["nodes"] > 0 and st["tris"] > 0
    assert st["max_stack"] <= 3 * b.max_depth   # a 4-wide step pushes up to three references
    cut = hcc.select_cut(d["bvh"], hcc.density(d["bvh"]), 1024, 32)
    keys = hcc.encode(d["diffuse"], cut)
    k_host = hcc.keys_to_numpy(keys)
    kept = keys.clone()
    perm = hcc.sort(keys, cut.info()["bits_used"])
    for p_dev, p_host in ((None, np.arange(k_host.shape[0])), (perm, _u32(perm))):
        ks = k_host[p_host]
        n_w = (ks.shape[0] + 31) // 32
        want = sum(len(np.unique(ks[32 * w:32 * w + 32])) for w in range(n_w)) / n_w
        assert abs(hcc.anc(kept, p_dev) - want) < 1e-9


# ------------------------------------------------------------------------------- pipeline
@pytest.mark.parametrize("name,K,bits", [("tiny", 64, 32), ("room_mid", 1024, 32), ("room_mid", 4096, 64)])
def test_pipeline_matches_stages(hcc, dev_cases, name, K, bits):
    import oracle
    d = dev_cases[name]
    case = d["case"]
    cut = hcc.select_cut(d["bvh"], hcc.density(d["bvh"]), K, bits)
    n_max = max(d["diffuse"].shape[0], d["shadow"].shape[0])
    pipe = hcc.Pipeline(n_max, 64, host_staging=True)
    with pytest.raises(hcc.HccError):
        pipe.stage_ms()                       # nothing timed yet
    pipe.set_timing(True)
    for batch, mode in (("diffuse", hcc.TRACE_CLOSEST), ("shadow", hcc.TRACE_ANY)):
        ref = hcc.trace(d["bvh"], d[batch], None, mode)
        for order in (hcc.ORDER_NOSORT, hcc.ORDER_TWOPOINT, hcc.ORDER_HCC):
            perm_out = torch.full((d[batch].shape[0],), -1, dtype=torch.int32, device="cuda")
            got = pipe.reorder_trace(d["bvh"], cut, order, d[batch], mode, key_bits=bits, perm_out=perm_out)
            assert torch.equal(got.view(torch.uint8), ref.view(torch.uint8))
            ms = pipe.stage_ms()
            assert ms["trace"] > 0
            if order == hcc.ORDER_HCC:
                tables, _, _ = oracle.select_cut(case.bvh.nodes, K, bits)
                want = oracle.sort(oracle.encode_hcc(getattr(case, batch), case.bvh.nodes, tables))
                assert np.array_equal(_u32(perm_out), want)
            # host-buffer form
            rays_h = torch.from_numpy(getattr(case, batch)).pin_memory()
            hits_h = torch.empty(ref.shape, dtype=ref.dtype).pin_memory()
            pipe.reorder_trace_host(d["bvh"], cut, order, rays_h, hits_h, mode, key_bits=bits)
            assert torch.equal(hits_h.view(torch.uint8), ref.cpu().view(torch.uint8))
    pipe.close()


@pytest.mark.parametrize("name,K,bits", [("tiny", 64, 32), ("room_mid", 1024, 32), ("room_mid", 4096, 64)])
def test_pipeline_pair_matches_two_calls(hcc, dev_cases, name, K, bits):
    """hcc_reorder_trace_pair (batch b's chain overlaps batch a's traversal by dependent launch) gives the hits of the
    separate calls, for the three orders, repeatedly (the chains of successive pairs reuse the pipeline's buffers), with
    an empty first or second batch, and with HCC_NO_PDL-style plain launches covered by the single-call tests."""
    d = dev_cases[name]
    cut = hcc.select_cut(d["bvh"], hcc.density(d["bvh"]), K, bits)
    ra, rb = d["diffuse"], d["shadow"]
    pipe = hcc.Pipeline(max(ra.shape[0], rb.shape[0]), 64, pair=True)
    with pytest.raises(hcc.HccError):      # a pipeline without the pair scratch refuses the call
        hcc.Pipeline(16, 64).reorder_trace_pair(d["bvh"], cut, hcc.ORDER_HCC, ra[:8], hcc.TRACE_CLOSEST, torch.empty((8, 4), device="cuda"),
                                                rb[:8], hcc.TRACE_ANY, torch.empty(8, dtype=torch.uint8, device="cuda"), key_bits=bits)
    ref_a = hcc.trace(d["bvh"], ra, None, hcc.TRACE_CLOSEST)
    ref_b = hcc.trace(d["bvh"], rb, None, hcc.TRACE_ANY)
    ha, hb = torch.empty_like(ref_a), torch.empty_like(ref_b)
    for rep in range(4):
        for order in (hcc.ORDER_HCC, hcc.ORDER_NOSORT, hcc.ORDER_TWOPOINT):
            ha.fill_(-1.0); hb.fill_(7)
            pipe.reorder_trace_pair(d["bvh"], cut, order, ra, hcc.TRACE_CLOSEST, ha, rb, hcc.TRACE_ANY, hb, key_bits=bits)
            assert torch.equal(ha.view(torch.int32), ref_a.view(torch.int32)) and torch.equal(hb, ref_b), (rep, order)
    # the batches the other way round, and one of them empty
    ha.fill_(-1.0); hb.fill_(7)
    pipe.reorder_trace_pair(d["bvh"], cut, hcc.ORDER_HCC, rb, hcc.TRACE_ANY, hb, ra, hcc.TRACE_CLOSEST, ha, key_bits=bits)
    assert torch.equal(ha.view(torch.int32), ref_a.view(torch.int32)) and torch.equal(hb, ref_b)
    empty = ra[:0]
    he = torch.empty((0, 4), dtype=torch.float32, device="cuda")
    hb.fill_(7)
    pipe.reorder_trace_pair(d["bvh"], cut, hcc.ORDER_HCC, empty, hcc.TRACE_CLOSEST, he, rb, hcc.TRACE_ANY, hb, key_bits=bits)
    assert torch.equal(hb, ref_b)
    ha.fill_(-1.0)
    pipe.reorder_trace_pair(d["bvh"], cut, hcc.ORDER_HCC, ra, hcc.TRACE_CLOSEST, ha, rb[:0], hcc.TRACE_ANY, hb[:0], key_bits=bits)
    assert torch.equal(ha.view(torch.int32), ref_a.view(torch.int32))
    pipe.close()


# ------------------------------------------------------------------------------- errors
def test_error_reporting(hcc, dev_cases):
    d = dev_cases["tiny"]
    had = hcc.density(d["bvh"])
    with pytest.raises(hcc.HccError) as e:
        hcc.select_cut(d["bvh"], had, 0, 32)
    assert e.value.status == -1 and "K" in str(e.value)
    with pytest.raises(hcc.HccError):
        hcc.select_cut(d["bvh"], had, 64, 20)
    cut = hcc.Cut(64)
    with pytest.raises(hcc.HccError):
        hcc.encode(d["diffuse"], cut)            # no selection yet
    keys = torch.zeros(9, dtype=torch.int32, device="cuda")
    with pytest.raises(hcc.HccError) as e:
        hcc.sort(keys[1:], 32)                    # 4-byte offset: misaligned
    assert e.value.status == -2
    with pytest.raises(hcc.HccError):
        hcc.sort(torch.zeros(8, dtype=torch.int32, device="cuda"), 40)
    with pytest.raises(hcc.HccError):
        hcc.trace(d["bvh"], d["diffuse"], None, 7)
    bad = d["case"].bvh.nodes.copy()
    bad["left_or_first"][0] = 0                   # child not after its parent
    with pytest.raises(hcc.HccError):
        hcc.Bvh(bad, d["case"].bvh.tris, d["case"].bvh.prim_idx)
    # n = 0 is a no-op everywhere
    empty = torch.zeros((0, 8), dtype=torch.float32, device="cuda")
    cut = hcc.select_cut(d["bvh"], had, 64, 32)
    assert hcc.encode(empty, cut).shape[0] == 0
    assert hcc.trace(d["bvh"], empty, None, hcc.TRACE_ANY).shape[0] == 0


# ----------------------------------------------------------------- (a4) edge cases of the traversal
def _rand_rays(n, seed, lo=-0.2, hi=1.2, axis_parallel=False):
    """Seeded rays with origins in [lo, hi]^3; with axis_parallel, directions have one or two
    exactly-zero components (the slab arithmetic's degenerate case)."""
    from hcc_inputs import rng as hrng
    u = hrng.u01(seed, 0, np.arange(n, dtype=np.uint64), np.arange(7, dtype=np.uint64)[:, None]).T
    rays = np.zeros((n, 8), dtype=np.float32)
    rays[:, 0:3] = lo + (hi - lo) * u[:, 0:3]
    d = 2.0 * u[:, 3:6] - 1.0
    if axis_parallel:
        kill = (u[:, 6] * 6).astype(np.int64)          # 0..5: which components to zero
        d[kill % 3 == 0, 0] = 0.0
        d[kill % 3 == 1, 1] = 0.0
        d[kill >= 3, 2] = 0.0
        d[np.abs(d).sum(axis=1) == 0, 0] = 1.0
        d[::7] = np.sign(d[::7]) * (d[::7] != 0)       # exact +-1 axis directions
        d[(np.abs(d).sum(axis=1) == 0)] = (0.0, -1.0, 0.0)
    d /= np.linalg.norm(d, axis=1, keepdims=True)
    rays[:, 4:7] = d
    rays[:, 3] = 0.0
    rays[:, 7] = np.inf
    return rays


def _check_trace_both_modes(hcc, b, rays):
    import oracle
    bvh = hcc.Bvh(b.nodes, b.tris, b.prim_idx)
    rd = torch.from_numpy(rays).cuda()
    want = oracle.closest_brute(rays, b.tris)
    got = hcc.hits_to_numpy(hcc.trace(bvh, rd, None, hcc.TRACE_CLOSEST))

    class _C:
        bvh = b
    check_closest(_C, rays, got, want)
    occ = hcc.trace(bvh, rd, None, hcc.TRACE_ANY).cpu().numpy()
    assert np.array_equal(occ, oracle.any_brute(rays, b.tris))
    return want


def test_trace_axis_parallel_rays_vs_brute_force(hcc, tiny):
    """Zero direction components: the quantised slab test must neither produce NaN culls nor
    miss a triangle (hits are defined by the triangle predicate alone)."""
    rays = _rand_rays(6000 + 13, 0xA11CE, axis_parallel=True)
    want = _check_trace_both_modes(hcc, tiny.bvh, rays)
    assert (~np.isinf(want[0])).sum() > 50


@pytest.mark.parametrize("dist", [30.0, 1000.0, 5000.0])
def test_trace_distant_origins_vs_brute_force(hcc, tiny, dist):
    """Origins `dist` scene extents away, aimed at points inside the scene: the slack of the
    quantised slab test grows with the origin's distance (include/hcc.h, hcc_trace), so no box
    holding a triangle the predicate accepts is culled.  (The triangle predicate itself is
    evaluated with the same coarse fp32 origin on both sides.)"""
    from hcc_inputs import rng as hrng
    n = 4000 + 7
    u = hrng.u01(0xFA4, int(dist), np.arange(n, dtype=np.uint64), np.arange(6, dtype=np.uint64)[:, None]).T
    target = (0.1 + 0.8 * u[:, 0:3]).astype(np.float32)
    d = 2.0 * u[:, 3:6] - 1.0
    d /= np.linalg.norm(d, axis=1, keepdims=True)
    rays = np.zeros((n, 8), dtype=np.float32)
    rays[:, 0:3] = target - np.float32(dist) * d.astype(np.float32)
    o = rays[:, 0:3].astype(np.float64)
    dd = target.astype(np.float64) - o                      # direction recomputed from the ROUNDED origin
    dd /= np.linalg.norm(dd, axis=1, keepdims=True)
    rays[:, 4:7] = dd
    rays[:, 3] = 0.0
    rays[:, 7] = np.inf
    want = _check_trace_both_modes(hcc, tiny.bvh, rays)
    assert (~np.isinf(want[0])).sum() > 50


def test_trace_many_launches_in_flight_on_two_streams(hcc, dev_cases):
    """More launches than work-counter slots (1024), alternating between two streams: every launch
    zeroes its own counter on its own stream, so results never depend on what ran before."""
    d = dev_cases["room_small"]
    ref = hcc.trace(d["bvh"], d["diffuse"], None, hcc.TRACE_CLOSEST)
    sub = d["diffuse"][:999].contiguous()
    streams = [torch.cuda.Stream(), torch.cuda.Stream()]
    outs = [torch.empty((999, 4), dtype=torch.float32, device="cuda") for _ in range(2)]
    torch.cuda.synchronize()
    for i in range(1100):
        with torch.cuda.stream(streams[i & 1]):
            hcc.trace(d["bvh"], sub, None, hcc.TRACE_CLOSEST, hits=outs[i & 1], stream=streams[i & 1])
    torch.cuda.synchronize()
    for o in outs:
        assert torch.equal(o.view(torch.int32), ref[:999].view(torch.int32))


def test_trace_flat_scene_vs_brute_force(hcc):
    """All triangles in the plane z = 0.25 (zero scene extent along z): the traversal grid is
    degenerate on that axis."""
    import hcc_inputs
    from hcc_inputs import rng as hrng
    n = 300
    u = hrng.u01(0xF1A7, 0, np.arange(n, dtype=np.uint64), np.arange(6, dtype=np.uint64)[:, None]).T
    tris = np.zeros((n, 3, 3), dtype=np.float32)
    c = u[:, 0:2]
    for k in range(3):
        tris[:, k, 0:2] = c + 0.05 * (u[:, 2 * k % 6:2 * k % 6 + 2] - 0.5)
    tris[:, :, 2] = 0.25
    b = hcc_inputs.build_bvh(tris)
    rays = np.concatenate([_rand_rays(3000, 0xF1A8, lo=0.0, hi=1.0), _rand_rays(1000, 0xF1A9, lo=0.0, hi=1.0, axis_parallel=True)])
    rays[:, 2] = np.where(np.arange(rays.shape[0]) % 2 == 0, 0.9, -0.4)      # above and below the plane
    want = _check_trace_both_modes(hcc, b, rays)
    assert (~np.isinf(want[0])).sum() > 20


def test_trace_root_leaf_bvh(hcc):
    """A BVH that is one leaf (<= 4 triangles): the leaf is wrapped in a wide node of its own (bvh.cu), so the traversal
    starts on a wide-node reference whose only child is the leaf."""
    import hcc_inputs
    tris = np.array([[[0, 0, 0], [1, 0, 0], [0, 1, 0]], [[0, 0, 0.5], [1, 0, 0.5], [0, 1, 0.5]]], dtype=np.float32)
    b = hcc_inputs.build_bvh(tris)
    assert b.n_nodes == 1
    rays = _rand_rays(257, 0x1EAF)
    rays[:, 0:3] = (0.2, 0.2, 1.0)
    _check_trace_both_modes(hcc, b, rays)


@pytest.mark.parametrize("scene", ["tiny", "room_small"])
def test_trace_leaves_of_up_to_eight_triangles(hcc, scene, tiny, room_small):
    """BVHs built with max_leaf = 8 (include/hcc.h admits leaf counts 1..8): a leaf of 5..8 triangles becomes a wide node
    of its own with two halves (bvh.cu), which no max_leaf = 4 tree exercises."""
    import hcc_inputs
    src = {"tiny": tiny, "room_small": room_small}[scene].bvh
    b = hcc_inputs.build_bvh(src.tris, max_leaf=8)
    counts = b.nodes["count"][b.nodes["count"] > 0]
    assert counts.max() > 4 and counts.max() <= 8
    lo, hi = b.nodes["lo"][0], b.nodes["hi"][0]
    rays = _rand_rays(20000 + 11, 0x8EAF)
    rays[:, 0:3] = lo + (hi - lo) * rays[:, 0:3]         # origins in and around the scene box
    want = _check_trace_both_modes(hcc, b, rays)
    assert (~np.isinf(want[0])).sum() > 1000


@pytest.mark.parametrize("n_tris", [5, 8])
def test_trace_single_leaf_of_five_and_eight_triangles_with_ties(hcc, n_tris):
    """A hand-made BVH that is ONE leaf of 5 or 8 triangles (the root leaf is split into two halves under a wide node).
    Triangles 1 and n_tris-1 are the same triangle, one in each half: the two tests give the same t, and the lowest
    prim id must win (include/hcc.h: "ties to the lowest prim id")."""
    import hcc_inputs
    import oracle
    base = np.array([[0.0, 0.0, 0.0], [1.0, 0.0, 0.0], [0.0, 1.0, 0.0]], dtype=np.float32)
    tris = np.stack([base + np.float32([0, 0, 0.1 * (k + 1)]) for k in range(n_tris)])
    tris[1] = tris[n_tris - 1] = base + np.float32([0, 0, 0.05])       # the nearest plane from below, twice
    b = hcc_inputs.make_bvh([((0, 0, 0.05), (1, 1, 0.1 * n_tris), 0, n_tris)], tris)
    rays = _rand_rays(513, 0x71E5)
    rays[:, 0:3] = (0.2, 0.2, -1.0)
    rays[:, 0:2] += 0.1 * rays[:, 4:6]
    rays[:, 4:7] = (0.0, 0.0, 1.0)
    want = _check_trace_both_modes(hcc, b, rays)
    bvh = hcc.Bvh(b.nodes, b.tris, b.prim_idx)
    t, prim, _, _ = hcc.hits_to_numpy(hcc.trace(bvh, torch.from_numpy(rays).cuda(), None, hcc.TRACE_CLOSEST))
    assert np.all(~np.isinf(t)) and np.all(prim == 1) and np.array_equal(prim, want[1])
    # from above the farthest plane is nearest; it is unique
    rays[:, 2] = 2.0
    rays[:, 6] = -1.0
    want = _check_trace_both_modes(hcc, b, rays)
    assert np.all(want[1] == n_tris - 2)


def test_pair_call_orders_later_work_behind_both_batches(hcc, dev_cases):
    """Work enqueued on the stream right after hcc_reorder_trace_pair sees the hits of BOTH batches.  The second traversal
    kernel is a dependent launch that does not wait at entry; it must still not complete before the first (it waits before
    exit).  Worst case: a long batch a and a tiny batch b, then a device-to-host copy of hits_a with nothing in between."""
    d = dev_cases["room_mid"]
    cut = hcc.select_cut(d["bvh"], hcc.density(d["bvh"]), 1024, 32)
    ra = d["diffuse"].repeat(8, 1).contiguous()          # 524,288 closest-hit rays
    rb = d["shadow"][:8].contiguous()
    ref_a = hcc.trace(d["bvh"], ra, None, hcc.TRACE_CLOSEST)
    ref_b = hcc.trace(d["bvh"], rb, None, hcc.TRACE_ANY)
    ha, hb = torch.empty_like(ref_a), torch.empty_like(ref_b)
    host_a = torch.empty(ref_a.shape, dtype=torch.float32).pin_memory()
    pipe = hcc.Pipeline(ra.shape[0], 64, pair=True)
    want = ref_a.cpu().view(torch.int32)
    for order in (hcc.ORDER_HCC, hcc.ORDER_NOSORT):
        for rep in range(5):
            ha.fill_(-1.0); hb.fill_(7); host_a.fill_(-2.0)
            pipe.reorder_trace_pair(d["bvh"], cut, order, ra, hcc.TRACE_CLOSEST, ha, rb, hcc.TRACE_ANY, hb)
            host_a.copy_(ha, non_blocking=True)          # directly behind the call, same stream
            torch.cuda.current_stream().synchronize()
            assert torch.equal(host_a.view(torch.int32), want), (order, rep)
            assert torch.equal(hb, ref_b)
    pipe.close()


def test_pipeline_synchronize_waits_for_the_last_call_of_any_form(hcc, dev_cases):
    """hcc_pipeline_synchronize after a host-buffer call followed by a device-buffer call waits for the LATTER (the host
    form's completion event must not be mistaken for it)."""
    d = dev_cases["room_mid"]
    cut = hcc.select_cut(d["bvh"], hcc.density(d["bvh"]), 1024, 32)
    rays_h = d["case"].diffuse[:4096]
    ra = d["diffuse"].repeat(16, 1).contiguous()         # about a millisecond of device work
    ha = torch.empty((ra.shape[0], 4), dtype=torch.float32, device="cuda")
    pipe = hcc.Pipeline(ra.shape[0], 64, host_staging=True)
    hits_h = np.empty((4096, 4), dtype=np.float32)
    s = torch.cuda.current_stream()
    for rep in range(5):
        pipe.reorder_trace_host(d["bvh"], cut, hcc.ORDER_HCC, rays_h, hits_h, hcc.TRACE_CLOSEST)
        pipe.reorder_trace(d["bvh"], cut, hcc.ORDER_HCC, ra, hcc.TRACE_CLOSEST, hits=ha)
        pipe.synchronize()
        assert s.query(), rep                            # nothing of the device call is still running
    pipe.close()


def test_trace_deep_chain_bvh_spills_the_stack(hcc):
    """A degenerate comb (depth 40) of nested boxes: every chain node has a small INTERNAL sibling (two
    one-triangle leaves) that is hit too and lies farther than the rest of the chain, so it is pushed at
    every level (leaves never go to the stack): the per-thread stack outgrows its shared-memory rows,
    spills to local memory and comes back."""
    import hcc_inputs
    depth = 40
    zs = [0.02 * (k + 1) for k in range(depth + 1)]
    tris = []
    for k in range(depth):          # S_k: two triangles side by side in the plane z_k
        tris.append([[0.1, 0.1, zs[k]], [0.5, 0.1, zs[k]], [0.1, 0.9, zs[k]]])
        tris.append([[0.5, 0.1, zs[k]], [0.9, 0.1, zs[k]], [0.5, 0.9, zs[k]]])
    tris.append([[0.1, 0.1, zs[depth]], [0.9, 0.1, zs[depth]], [0.1, 0.9, zs[depth]]])
    # chain node I_k at 2k (children S_k at 2k+1 and I_{k+1} at 2k+2); the last chain node (2*depth) is a leaf;
    # the two leaves of S_k follow at 2*depth + 1 + 2k
    nodes = [None] * (2 * depth + 1 + 2 * depth)
    for k in range(depth):
        nodes[2 * k] = ((0.1, 0.1, zs[k]), (0.9, 0.9, zs[depth]), 2 * k + 1, 0)
        nodes[2 * k + 1] = ((0.1, 0.1, zs[k]), (0.9, 0.9, zs[k]), 2 * depth + 1 + 2 * k, 0)
        nodes[2 * depth + 1 + 2 * k] = ((0.1, 0.1, zs[k]), (0.5, 0.9, zs[k]), 2 * k, 1)
        nodes[2 * depth + 2 + 2 * k] = ((0.5, 0.1, zs[k]), (0.9, 0.9, zs[k]), 2 * k + 1, 1)
    nodes[2 * depth] = ((0.1, 0.1, zs[depth]), (0.9, 0.9, zs[depth]), 2 * depth, 1)
    b = hcc_inputs.make_bvh(nodes, np.array(tris, dtype=np.float32))
    assert b.max_depth == depth + 1
    # rays travelling in -z from above meet the LAST plane first: the nearest child is always the rest of
    # the chain, so the small internal siblings on the way down are all pushed
    rays = _rand_rays(2000 + 5, 0xDEE9, lo=0.0, hi=1.0)
    rays[:, 2] = 2.0
    rays[:, 4:7] = (0.0, 0.0, -1.0)
    rays[1::2, 4:7] = (0.05, -0.03, -1.0)
    rays[1::2, 4:7] /= np.linalg.norm(rays[1::2, 4:7], axis=1, keepdims=True)
    bvh = hcc.Bvh(b.nodes, b.tris, b.prim_idx)
    st = hcc.trace_stats(bvh, torch.from_numpy(rays).cuda(), None, hcc.TRACE_CLOSEST)
    assert st["max_stack"] > 16, st
    _check_trace_both_modes(hcc, b, rays)


@pytest.mark.parametrize("n", [1, 31, 32, 33, 127, 129, 4097])
def test_trace_ragged_sizes_and_counter_rearm(hcc, dev_cases, n):
    """Ragged batch sizes, and > 256 launches on one BVH (the work-counter slots are reused and
    must have re-armed themselves)."""
    d = dev_cases["room_small"]
    ref = hcc.trace(d["bvh"], d["diffuse"], None, hcc.TRACE_CLOSEST)
    sub = d["diffuse"][:n].contiguous()
    reps = 300 if n == 33 else 3
    for _ in range(reps):
        got = hcc.trace(d["bvh"], sub, None, hcc.TRACE_CLOSEST)
    assert torch.equal(got.view(torch.int32), ref[:n].view(torch.int32))
