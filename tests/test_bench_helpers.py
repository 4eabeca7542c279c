"""Host logic of bench.py (no GPU): the sort's byte models and the ncu-traffic look-up that refuses stale captures."""
import importlib
import os
import sys

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)


def _bench():
    return importlib.import_module("bench")


def test_sort_byte_models():
    b = _bench()
    # (SURVEY.md 8(d) bytes, bytes the kernels move): first pass reads no ids, last pass writes no keys
    assert b.sort_bytes(4, 4) == (68, 60)
    assert b.sort_bytes(8, 6) == (152, 140)
    assert b.sort_bytes(8, 8) == (200, 188)
    assert b.sort_bytes(4, 1) == (20, 12)          # one pass: histogram read + key read + id write
    assert b.sort_bytes(4, 2) == (36, 28)
    assert b.sort_bytes(4, 0) == (0, 0)


def test_ncu_traffic_is_keyed_by_the_kernel_sources(tmp_path, monkeypatch):
    b = _bench()
    h = b.kernel_source_hash()
    assert len(h) == 16 and h == b.kernel_source_hash()
    f = tmp_path / "traffic.md"
    f.write_text("# header\n"
                 f"traffic room diffuse dram_read_bytes=100 dram_write_bytes=23 duration_us=1.0 sources={h}\n"
                 "traffic room shadow dram_read_bytes=5 dram_write_bytes=6 duration_us=1.0 sources=0123456789abcdef\n")
    monkeypatch.setattr(b, "TRAFFIC_FILE", str(f))
    assert b.ncu_traffic("room", "diffuse") == 123.0
    assert b.ncu_traffic("room", "shadow") is None        # captured from other sources: never quoted
    assert b.ncu_traffic("fig1", "diffuse") is None       # no line
    monkeypatch.setattr(b, "TRAFFIC_FILE", str(tmp_path / "missing.md"))
    assert b.ncu_traffic("room", "diffuse") is None
