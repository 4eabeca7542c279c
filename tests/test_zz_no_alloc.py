"""hcc_sort_static, the sort entry point for callers that cannot allocate device memory.

Who needs it: code that runs inside somebody else's GPU process and is handed only its input and output
buffers (a renderer plug-in under a host application that owns the memory pool), or code on a path where a
cudaMalloc is not acceptable (a frame loop that must not block on the driver's allocation lock, a process
whose HBM is already fully committed).  hcc_sort asks such a caller for a workspace it has no way to
provide; hcc_sort_static keeps a fixed 4 MiB workspace inside the library instead and is limited to
262,144 pairs per call.

The checks below compare it with hcc_sort on the same keys: the permutation must be identical (the bar of
every sort test in this suite is bit-exact), on two calls in a row, because the shared workspace still holds
the first call's histograms, tickets and status rows when the second call starts.

This file is named so that pytest collects it last: under `pytest -x` a failure here cannot hide the
results of the parity tests.  It must pass alone in a fresh process (its first call then performs the
per-device set-up) and after the rest of the suite.
"""
import ctypes

import numpy as np
import pytest

torch = pytest.importorskip("torch")


@pytest.fixture(scope="module")
def hcc():
    if not torch.cuda.is_available():
        pytest.skip("no CUDA device")
    import paper_2305_16652_b200 as h
    return h


def _keys(rng, n, cb, bits_used):
    k = rng.integers(0, (1 << bits_used) - 1, size=n, dtype=np.uint64, endpoint=True)
    k[rng.uniform(size=n) < 0.3] = k[0]            # long runs of equal keys: stability matters
    dt = np.uint32 if cb == 32 else np.uint64
    return torch.from_numpy(k.astype(dt).view(np.int32 if cb == 32 else np.int64))


@pytest.mark.gpu
@pytest.mark.parametrize("cb,bits_used", [(32, 32), (32, 20), (64, 64), (64, 40)])
def test_sort_static_equals_sort_on_two_calls_in_a_row(hcc, cb, bits_used):
    rng = np.random.default_rng(1000 + cb + bits_used)
    # the second call is SMALLER than the first and of different shape: it uses fewer status rows and fewer
    # passes' worth of the control region, so anything it failed to clear would still hold the first call's values
    sizes = [hcc.SORT_STATIC_MAX_N, 100003, 4097]
    for n in sizes:
        k = _keys(rng, n, cb, bits_used).cuda()
        want = hcc.sort(k.clone(), bits_used)                  # the existing path, workspace from torch
        perm = torch.full((n,), -1, dtype=torch.int32, device="cuda")
        got = hcc.sort_static(k.clone(), bits_used, perm)      # back to back on the same stream: no overlap
        assert got.data_ptr() == perm.data_ptr()
        assert torch.equal(got, want), (n, cb, bits_used)
    # and the same input twice in a row gives the same answer twice
    k = _keys(rng, 65536 + 7, cb, bits_used).cuda()
    want = hcc.sort(k.clone(), bits_used)
    for _ in range(2):
        perm = torch.empty(k.shape[0], dtype=torch.int32, device="cuda")
        assert torch.equal(hcc.sort_static(k.clone(), bits_used, perm), want)


@pytest.mark.gpu
def test_sort_static_uses_no_device_memory_of_its_own(hcc):
    """The free-memory figure of the driver does not move across calls (after one warm-up call that does the
    per-device set-up); inputs and outputs are allocated beforehand."""
    rng = np.random.default_rng(7)
    k = _keys(rng, hcc.SORT_STATIC_MAX_N, 64, 64).cuda()
    perm = torch.empty(k.shape[0], dtype=torch.int32, device="cuda")
    copies = [k.clone() for _ in range(4)]
    hcc.sort_static(copies[0], 64, perm)
    torch.cuda.synchronize()
    free0, _ = torch.cuda.mem_get_info()
    for c in copies[1:]:
        hcc.sort_static(c, 64, perm)
    torch.cuda.synchronize()
    free1, _ = torch.cuda.mem_get_info()
    assert free1 == free0


def test_sort_static_rejects_sizes_beyond_its_limit():
    """Argument checks come before any CUDA call, so this runs without a GPU.  Nothing is dereferenced."""
    import paper_2305_16652_b200 as h
    L = h.lib()
    dummy = ctypes.c_void_p(256)
    assert L.hcc_sort_static(dummy, h.SORT_STATIC_MAX_N + 1, 32, 32, dummy, None) == -5
    msg = L.hcc_last_error()
    assert b"262144" in msg and b"hcc_sort" in msg
    assert L.hcc_sort_static(dummy, 16, 48, 32, dummy, None) == -1
    assert L.hcc_sort_static(dummy, 16, 32, 40, dummy, None) == -1
    assert L.hcc_sort_static(None, 0, 32, 32, None, None) == 0     # n = 0 is a no-op, as everywhere
