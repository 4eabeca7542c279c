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


def test_final_line_is_compact_and_carries_the_contract():
    """The driver parses the LAST stdout line and keeps only the tail of stdout: the line must stay under 4 KB whatever
    the optional sections hold (round 2's 39 KB line was not parsed)."""
    import json
    b = _bench()
    stage = lambda ms, bound, frac: {"ms": ms, "bound": bound, "achieved": 1234.56789, "peak": 6535.1, "unit": "GB/s", "frac": frac,
                                     "passes": 4, "bytes_per_pair_moved": 60, "alu_frac_by_ops_per_test": {"26": 0.9, "20": 0.7, "14": 0.5}}
    stages = {bn: {"encode": stage(0.0312345678, "hbm", 0.1712345), "sort": stage(0.0451234, "hbm", 0.2812345),
                   "trace": stage(0.3571234, "alu", 0.1661234)} for bn in ("diffuse", "shadow")}
    big = {f"cell_{i}": {"encode_ms": 0.123456789, "sort_ms": 0.2, "trace_ms": 0.3, "note": "x" * 50} for i in range(400)}
    full = {"metric": b.METRIC, "value": 3566.123456789, "unit": b.UNIT, "n_gpus": 1, "steps": 100, "warmup": 3,
            "ms_per_step": 0.882123456, "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f32",
            "data": "synthetic",
            "config": {"workload": "config 2 'room' of BASELINE.json", "triangles": 64012, "bvh_nodes": 42000, "K": 1024, "key_bits": 32,
                       "diffuse_rays": 1048576, "shadow_rays": 2097152, "resolution": "512x512x4spp", "bounce": 1,
                       "l2": "flushed between timed steps (256 MiB write)", "parallelism": "p" * 260,
                       "lib": "paper_2305_16652_b200/libhcc_b200.so", "no_pdl": False},
            "clocks": {"sm_mhz": 1965.0, "sm_max_mhz": 1965.0, "reasons": [], "samples": 12},
            "e2e": {"value": 1456.123, "unit": b.UNIT, "ms_per_step": 2.16, "h2d_bytes_per_step": 100663296,
                    "d2h_bytes_per_step": 18874368, "how": "h" * 120},
            "gpu_launches": 1800,
            "roofline": {"bound": "alu", "achieved": 6.18, "peak": 37.22, "unit": "Tlaneop/s", "frac": 0.1661, "traffic": 83800000.0,
                         "traffic_unit": "t" * 160, "kernel": "trace (shadow batch)", "peak_source": "s" * 60},
            "cpu_baseline": {"value": 0.361, "unit": b.UNIT, "cores": 1, "kind": "oracle", "sample": "s" * 150,
                             "split_s": {"encode": 1.0, "sort": 0.5, "trace": 20.0}, "host_cores": 16},
            "cut": {"widths": [32, 32], "K_eff": 1024, "bits_used": 32, "container_bits": 32, "cut_ms": 0.5},
            "speedup_hcc": {"diffuse": {"incl_vs_nosort": 0.8}, "shadow": {"incl_vs_nosort": 0.8}, "pair_incl_vs_nosort": 0.81,
                            "pair_incl_vs_twopoint": 1.0, "all_incl_vs_nosort": 0.79, "all_incl_vs_twopoint": 0.97},
            "stages_roofline_hcc": stages,
            "orders": big, "studies": big, "other_configs": big, "diagnostics": big, "speedup_hcc_by_bounce": big}
    line = b.final_line(full)
    assert "\n" not in line and len(line) < 4096
    got = json.loads(line)
    for k in ("metric", "value", "unit", "n_gpus", "steps", "warmup", "ms_per_step", "higher_is_better", "scaling", "dtype", "data",
              "config", "clocks", "e2e", "gpu_launches", "roofline", "cpu_baseline", "cut", "speedup_hcc", "stages_roofline_hcc"):
        assert k in got, k
    assert got["value"] > 0 and got["roofline"]["frac"] == 0.1661 and got["roofline"]["traffic"] == 83800000.0
    assert got["e2e"]["h2d_bytes_per_step"] == 100663296 and got["e2e"]["d2h_bytes_per_step"] == 18874368
    assert got["cpu_baseline"]["kind"] == "oracle" and got["cpu_baseline"]["cores"] == 1
    assert set(got["speedup_hcc"]) == {"pair_incl_vs_nosort", "pair_incl_vs_twopoint", "all_incl_vs_nosort", "all_incl_vs_twopoint"}
    assert got["stages_roofline_hcc"]["shadow"]["trace"] == {"ms": 0.35712, "bound": "alu", "frac": 0.16612}
    for k in ("orders", "studies", "other_configs", "diagnostics", "speedup_hcc_by_bounce"):
        assert k not in got
    # free text that would push the line over the limit is cut, never the numbers
    full["cpu_baseline"]["sample"] = "s" * 3000
    line2 = b.final_line(full)
    assert len(line2) < 4096 and json.loads(line2)["cpu_baseline"]["value"] == 0.361


def test_default_run_is_the_headline_only():
    """Studies, other configs, later bounces and the large-batch legs are opt-in (bench.py --help)."""
    src = open(os.path.join(ROOT, "bench.py")).read()
    assert '"--configs", default=""' in src
    assert 'ap.add_argument("--studies", action="store_true",\n' in src
    assert "default=True" not in src.split("def main()")[1]
