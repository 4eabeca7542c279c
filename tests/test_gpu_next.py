"""Parity of the CUDA path against the oracle for the NEXT rows of the scope table
(SURVEY.md §8(f)): f1 sort truncation, f3 prefix path code, f4 regular grid encoding.
Keys, boxes and permutations are bit-exact."""
import numpy as np
import pytest

pytestmark = pytest.mark.gpu

torch = pytest.importorskip("torch")


@pytest.fixture(scope="module")
def hcc():
    if not torch.cuda.is_available():
        pytest.skip("no CUDA device")
    import paper_2305_16652_b200 as h
    return h


@pytest.fixture(scope="module")
def cases(hcc, tiny, room_mid):
    out = {}
    for name, case in (("tiny", tiny), ("room_mid", room_mid)):
        b = case.bvh
        out[name] = dict(case=case, bvh=hcc.Bvh(b.nodes, b.tris, b.prim_idx),
                         diffuse=torch.from_numpy(case.diffuse).cuda(), shadow=torch.from_numpy(case.shadow).cuda())
    return out


# ------------------------------------------------------------------------------- f1
@pytest.mark.parametrize("cb,used", [(32, 32), (32, 20), (64, 48), (64, 64)])
@pytest.mark.parametrize("bit_lo", [0, 3, 8, 16, 29])
@pytest.mark.parametrize("n", [1, 4097, 100003])
def test_sort_range_vs_oracle(hcc, cb, used, bit_lo, n):
    import oracle
    bit_lo = min(bit_lo, used)
    g = torch.Generator(device="cpu").manual_seed(1234 + n + used)
    k = torch.randint(0, 2 ** 62, (n,), generator=g, dtype=torch.int64) & ((1 << used) - 1)
    k[::5] = k[0]
    keys_h = k.numpy().astype(np.uint64)
    keys = k.cuda() if cb == 64 else torch.from_numpy(keys_h.astype(np.uint32).view(np.int32)).cuda()
    perm = hcc.sort(keys, used, bit_lo=bit_lo)
    want = oracle.sort_from_bit(keys_h, bit_lo)
    assert np.array_equal(perm.cpu().numpy().view(np.uint32), want)


def test_pipeline_sort_skip_bits(hcc, cases):
    """hcc_pipeline_set_sort_skip_bits: the pipeline's permutation is the truncated sort's, and the
    hits do not depend on the order."""
    import oracle
    d = cases["room_mid"]
    cut = hcc.select_cut(d["bvh"], hcc.density(d["bvh"]), 1024, 32)
    used = cut.info()["bits_used"]
    keys_h = hcc.keys_to_numpy(hcc.encode(d["diffuse"], cut)).astype(np.uint64)
    n = d["diffuse"].shape[0]
    pipe = hcc.Pipeline(n, 64)
    ref = hcc.trace(d["bvh"], d["diffuse"], None, hcc.TRACE_CLOSEST)
    for skip in (0, 8, 16, used, 40):
        pipe.set_sort_skip_bits(skip)
        perm = torch.empty(n, dtype=torch.int32, device="cuda")
        hits = pipe.reorder_trace(d["bvh"], cut, hcc.ORDER_HCC, d["diffuse"], hcc.TRACE_CLOSEST, perm_out=perm)
        assert np.array_equal(perm.cpu().numpy().view(np.uint32), oracle.sort_from_bit(keys_h, min(skip, used)))
        assert torch.equal(hits.view(torch.int32), ref.view(torch.int32))


# ------------------------------------------------------------------------------- f3
@pytest.mark.parametrize("name", ["tiny", "room_mid"])
@pytest.mark.parametrize("bits", [16, 24, 32, 48, 64])
def test_ppc_keys_bit_exact(hcc, cases, name, bits):
    import oracle
    d = cases[name]
    b = d["case"].bvh
    for batch in ("diffuse", "shadow"):
        rays_h = getattr(d["case"], batch)[:30011]
        got = hcc.keys_to_numpy(hcc.encode_ppc(d["bvh"], torch.from_numpy(rays_h).cuda(), bits)).astype(np.uint64)
        want = oracle.encode_ppc(rays_h, b.nodes, bits)
        assert np.array_equal(got, want)
        assert len(np.unique(want)) > 8


def test_ppc_root_leaf_and_errors(hcc):
    import hcc_inputs
    import oracle
    tris = np.array([[[0, 0, 0], [1, 0, 0], [0, 1, 0]]], dtype=np.float32)
    b = hcc_inputs.build_bvh(tris)
    bvh = hcc.Bvh(b.nodes, b.tris, b.prim_idx)
    rays = np.zeros((64, 8), np.float32)
    rays[:, 0:3] = (0.2, 0.2, 1.0); rays[:, 6] = -1.0; rays[:, 7] = np.inf
    rays[32:, 0] = 5.0
    got = hcc.keys_to_numpy(hcc.encode_ppc(bvh, torch.from_numpy(rays).cuda(), 16)).astype(np.uint64)
    assert np.array_equal(got, oracle.encode_ppc(rays, b.nodes, 16))
    assert set(got.tolist()) == {0, 1 << 15}
    with pytest.raises(hcc.HccError):
        hcc.encode_ppc(bvh, torch.from_numpy(rays).cuda(), 20)
    assert hcc.encode_ppc(bvh, torch.zeros((0, 8), dtype=torch.float32, device="cuda"), 32).shape[0] == 0


# ------------------------------------------------------------------------------- f4
@pytest.mark.parametrize("name", ["tiny", "room_mid"])
@pytest.mark.parametrize("widths,bits", [([8], 16), ([16, 16], 32), ([16, 8, 8], 32), ([32, 32], 64), ([4, 4, 4, 4], 16),
                                         ([16, 16, 16], 64)])
def test_grid_boxes_and_keys_bit_exact(hcc, cases, name, widths, bits):
    import oracle
    d = cases[name]
    cut = hcc.select_grid(d["bvh"], widths, bits)
    boxes, cnt = oracle.grid_tables(d["bvh"].scene_lo, d["bvh"].scene_hi, widths)
    ent, got_cnt = cut.read()
    assert np.array_equal(got_cnt, cnt) and np.all(ent == 0xFFFFFFFF)
    assert np.array_equal(cut.read_boxes().view(np.uint32), boxes.view(np.uint32))
    assert cut.info()["bits_used"] == sum(widths)
    for batch in ("diffuse", "shadow"):
        rays_h = getattr(d["case"], batch)[:40009]
        got = hcc.keys_to_numpy(hcc.encode(torch.from_numpy(rays_h).cuda(), cut)).astype(np.uint64)
        want = oracle.encode_tables(rays_h, boxes, widths, cnt)
        assert np.array_equal(got, want)


def test_grid_pipeline_and_errors(hcc, cases):
    """A grid cut drives the unchanged pipeline (encode -> sort -> trace); bad widths are refused."""
    import oracle
    d = cases["room_mid"]
    widths = [16, 8, 8]
    cut = hcc.select_grid(d["bvh"], widths, 32)
    boxes, cnt = oracle.grid_tables(d["bvh"].scene_lo, d["bvh"].scene_hi, widths)
    n = d["shadow"].shape[0]
    pipe = hcc.Pipeline(n, 64)
    perm = torch.empty(n, dtype=torch.int32, device="cuda")
    hits = pipe.reorder_trace(d["bvh"], cut, hcc.ORDER_HCC, d["shadow"], hcc.TRACE_ANY, perm_out=perm)
    keys = oracle.encode_tables(d["case"].shadow, boxes, widths, cnt)
    assert np.array_equal(perm.cpu().numpy().view(np.uint32), oracle.sort(keys))
    assert torch.equal(hits, hcc.trace(d["bvh"], d["shadow"], None, hcc.TRACE_ANY))
    for bad, bits in (([3], 16), ([16, 16, 16], 32), ([1], 16)):
        with pytest.raises(hcc.HccError):
            hcc.select_grid(d["bvh"], bad, bits)


# ------------------------------------------------------------------ host-buffer path, asynchronous form
def test_reorder_trace_host_async_matches_the_device_path(hcc, cases):
    """hcc_reorder_trace_host_async on two pipelines / two streams (bench.py's e2e leg) returns the
    same bytes as the device-buffer call."""
    d = cases["room_mid"]
    cut = hcc.select_cut(d["bvh"], hcc.density(d["bvh"]), 1024, 32)
    n_d, n_s = d["diffuse"].shape[0], d["shadow"].shape[0]
    pa, pb = hcc.Pipeline(n_d, 64, host_staging=True), hcc.Pipeline(n_s, 64, host_staging=True)
    sa, sb = torch.cuda.Stream(), torch.cuda.Stream()
    rays_a = torch.from_numpy(d["case"].diffuse).pin_memory()
    rays_b = torch.from_numpy(d["case"].shadow).pin_memory()
    hits_a = torch.empty((n_d, 4), dtype=torch.float32).pin_memory()
    hits_b = torch.empty(n_s, dtype=torch.uint8).pin_memory()
    torch.cuda.synchronize()
    pa.set_timing(True)
    for _ in range(3):
        hits_a.zero_(); hits_b.zero_()
        pa.reorder_trace_host_async(d["bvh"], cut, hcc.ORDER_HCC, rays_a, hits_a, hcc.TRACE_CLOSEST, stream=sa)
        pb.reorder_trace_host_async(d["bvh"], cut, hcc.ORDER_HCC, rays_b, hits_b, hcc.TRACE_ANY, stream=sb)
        pa.synchronize(); pb.synchronize()
        ref_a = hcc.trace(d["bvh"], d["diffuse"], None, hcc.TRACE_CLOSEST)
        ref_b = hcc.trace(d["bvh"], d["shadow"], None, hcc.TRACE_ANY)
        assert torch.equal(hits_a.cuda().view(torch.int32), ref_a.view(torch.int32))
        assert torch.equal(hits_b.cuda(), ref_b)
    ms = pa.stage_ms()
    assert ms["h2d"] > 0 and ms["trace"] > 0


# ------------------------------------------------------------------ f4: Algorithm 3 as printed (discard)
@pytest.mark.parametrize("name", ["tiny", "room_mid"])
@pytest.mark.parametrize("widths,bits", [([8, 8], 16), ([16, 8, 8], 32), ([4, 4, 4], 16), ([16, 16, 16], 64), ([32], 32)])
def test_alg3_discard_tables_and_keys_bit_exact(hcc, cases, name, widths, bits):
    import oracle
    d = cases[name]
    b = d["case"].bvh
    had = hcc.density(d["bvh"])
    cut = hcc.select_cut_levels(d["bvh"], had, widths, bits, flags=hcc.CUT_ALG3_DISCARD)
    want = oracle.level_tables(b.nodes, oracle.had(b.nodes), widths, discard=True)
    ent, cnt = cut.read()
    assert np.array_equal(cnt, want.table_cnt)
    assert np.array_equal(ent, want.entry_node)
    rays_h = d["case"].diffuse[:20011]
    got = hcc.keys_to_numpy(hcc.encode(torch.from_numpy(rays_h).cuda(), cut)).astype(np.uint64)
    assert np.array_equal(got, oracle.encode_hcc(rays_h, b.nodes, want))
    # the flag is per selection: the same handle re-selected without it gives reading R4's tables again
    hcc.select_cut_levels(d["bvh"], had, widths, bits, cut=cut)
    ent2, cnt2 = cut.read()
    kept = oracle.level_tables(b.nodes, oracle.had(b.nodes), widths)
    assert np.array_equal(ent2, kept.entry_node) and np.array_equal(cnt2, kept.table_cnt)
    with pytest.raises(hcc.HccError):
        hcc.select_cut_levels(d["bvh"], had, widths, bits, flags=6)


def test_plain_launches_give_the_same_results():
    """HCC_NO_PDL=1 turns every chained / overlapping launch into a plain one (the library's A/B switch, read once per
    process): the pair call and the single calls still agree with the default build's hits, bit for bit."""
    import os
    import subprocess
    import sys
    root = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
    code = r'''
import sys, hashlib
sys.path.insert(0, %r)
import numpy as np, torch, hcc_inputs, oracle
import paper_2305_16652_b200 as hcc
w = hcc_inputs.Workload("tiny")
b = w.bvh
def tc(bvh, rays):
    t, p, _, _ = oracle.closest_bvh(rays, bvh.nodes, bvh.prim_idx, bvh.tris); return t, p
d, s = w.first_bounce(tc)
bvh = hcc.Bvh(b.nodes, b.tris, b.prim_idx)
cut = hcc.select_cut(bvh, hcc.density(bvh), w.K, w.key_bits)
rd, rs = torch.from_numpy(d).cuda(), torch.from_numpy(s).cuda()
pipe = hcc.Pipeline(rs.shape[0], 64, pair=True)
hd = torch.empty((rd.shape[0], 4), dtype=torch.float32, device="cuda"); hs = torch.empty(rs.shape[0], dtype=torch.uint8, device="cuda")
for _ in range(3):
    pipe.reorder_trace_pair(bvh, cut, hcc.ORDER_HCC, rd, hcc.TRACE_CLOSEST, hd, rs, hcc.TRACE_ANY, hs)
one_d = pipe.reorder_trace(bvh, cut, hcc.ORDER_HCC, rd, hcc.TRACE_CLOSEST)
one_s = pipe.reorder_trace(bvh, cut, hcc.ORDER_HCC, rs, hcc.TRACE_ANY)
assert torch.equal(one_d.view(torch.uint8), hd.view(torch.uint8)) and torch.equal(one_s, hs)
print("DIGEST", hashlib.sha256(hd.cpu().numpy().tobytes() + hs.cpu().numpy().tobytes()).hexdigest())
''' % root
    digests = []
    for no_pdl in ("0", "1"):
        env = dict(os.environ, HCC_NO_PDL=no_pdl)
        r = subprocess.run([sys.executable, "-c", code], capture_output=True, text=True, env=env, timeout=600, cwd=root)
        assert r.returncode == 0, r.stderr[-2000:]
        digests.append([l for l in r.stdout.splitlines() if l.startswith("DIGEST")][-1])
    assert digests[0] == digests[1]
