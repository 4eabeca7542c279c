"""bench.py — the hot path of hierarchy-cut-code ray reordering on B200, measured.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--impl ours|reference] [--workload room|fig1|tiny]

One STEP = one pass of the whole per-batch hot path (Figure 11) over one
bounce of BASELINE.json config 2 ("room": 64,012 triangles, 512x512x4 spp): the diffuse batch
(1,048,576 closest-hit rays) and the shadow batch (2,097,152 any-hit rays), each
key-computed (hcc_encode), sorted (hcc_sort) and traced through the sorted indices (hcc_trace),
both in ONE C-ABI call, hcc_reorder_trace_pair (the kernels of the call are chained by programmatic
dependent launch; the per-stage split comes from separate, event-ordered hcc_reorder_trace calls).
Metric: secondary Mrays/s INCLUDING encode + sort.
The same rays are also run in the NoSort and TwoPoint orders and the
per-stage split, speed-ups, ANC and roofline fractions are reported in the
JSON line.  The cut (hcc_density + hcc_select_cut) is a once-per-scene pre-process in the
paper (:157, :218); it is timed separately ("cut_ms").

Inputs are seeded and synthetic (hcc_inputs/); the primaries are
traced by the library's own tracer (parity-tested against the oracle in tests/).  L2 is
flushed between timed steps (the batches, 100 MB, would otherwise sit in the 126 MB L2).

--impl reference times the CPU oracle (oracle/, single-threaded C) on a bounded sample of the
same workload; it is the only mode, with the cpu_baseline leg, that touches oracle/.
"""
import argparse
import json
import os
import subprocess
import sys
import threading
import time

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

import numpy as np

METRIC = "secondary Mrays/s incl. encode+sort (hierarchy cut code order; diffuse + shadow batches of one bounce)"
UNIT = "Mrays/s"

# Algorithmic work per ray, stated in DESIGN.md "Rooflines":
#  encode: 32 B ray read + key write;  sort: one histogram read + per pass read+write of (key, id)
#  trace : lane-operations = 68 per wide-node record fetched (four quantised child boxes: 24 cell->float
#          conversions, 24 fma, 16 min/max, 4 compares, trace.cu) + 36 per triangle test (the formula in
#          include/hcc.h); encode: 26 per exact fp32 slab test AS DEFINED (6 sub, 6 mul, 12 min/max, compare, bit); the kernel's
#          oriented form of the test executes 20 of them (no per-axis min/max), so alu_frac is algorithmic work over peak.
OPS_BOX, OPS_NODE, OPS_TRI = 26, 68, 36
# the same operations weighted by the issue cycles their pipe takes (B300_MICROARCH.md: min/max, compare, select, PRMT run on the
# ALU pipe at 16 lanes per scheduler and clock = 2 cycles per warp instruction; fma/mul/add at 1): per wide record 44 ALU-pipe
# operations + 24 fma = 112 issue cycles' worth; per triangle test 10 compares/selects + 26 fma/mul/add = 46
CYC_NODE, CYC_TRI = 2 * 44 + 24, 2 * 10 + 26
SM_COUNT, LANES_PER_SM = 148, 128
TRAFFIC_FILE = os.path.join(ROOT, "profiles", "r3_trace_traffic.md")
KERNEL_SOURCES = ("paper_2305_16652_b200/csrc/trace.cu", "paper_2305_16652_b200/csrc/bvh.cu",
                  "paper_2305_16652_b200/csrc/common.cuh")


def sort_bytes(key_b, passes):
    """Bytes per pair the sort moves through HBM: (algorithmic per SURVEY.md 8(d), what the kernels really move).
    Algorithmic: one histogram read + per pass a read and a write of (key, id).  Real: the first pass reads no ids
    (it synthesises them) and the last pass writes no keys (sort.cu)."""
    algo = key_b + passes * 2 * (key_b + 4)
    if passes == 0:
        return 0, 0
    if passes == 1:
        real = key_b + key_b + 4
    else:
        real = key_b + (2 * key_b + 4) + (passes - 2) * 2 * (key_b + 4) + (key_b + 8)
    return algo, real


def kernel_source_hash():
    """sha256 over the traversal kernel's sources: profiles/r3_trace_traffic.md records the hash its ncu capture
    was taken at, so a stale capture is never reported (the GPU box has no .git to ask for HEAD)."""
    import hashlib
    h = hashlib.sha256()
    for rel in KERNEL_SOURCES:
        with open(os.path.join(ROOT, rel), "rb") as f:
            h.update(f.read())
    return h.hexdigest()[:16]


def ncu_traffic(workload, batch):
    """dram__bytes_read.sum + dram__bytes_write.sum per launch of the trace kernel from the tracked ncu summary, or
    None when the file is missing, holds no line for this workload/batch or was captured from other sources."""
    try:
        want = kernel_source_hash()
        with open(TRAFFIC_FILE) as f:
            for line in f:
                t = line.split()
                if len(t) >= 6 and t[0] == "traffic" and t[1] == workload and t[2] == batch:
                    kv = dict(x.split("=", 1) for x in t[3:] if "=" in x)
                    if kv.get("sources") != want:
                        return None
                    return float(kv["dram_read_bytes"]) + float(kv["dram_write_bytes"])
    except Exception:
        return None
    return None


def _peaks():
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    try:
        with open(p) as f:
            d = json.load(f)
        return float(d["hbm_gbs"]), float(d.get("sm_max_mhz", 1965.0)), "measured"
    except Exception:
        return 6650.0, 1965.0, "fallback"


# ---- the final stdout line.  The driver keeps only the tail of stdout, so the LAST line is one compact JSON object
# (under 4 KB); everything else (per-order splits, later bounces, other configs, studies, counters) is printed as
# separate {"section": ...} lines BEFORE it, and only when asked for by flag, or written to --full-json.
FINAL_KEYS = ("metric", "value", "unit", "n_gpus", "steps", "warmup", "ms_per_step", "higher_is_better", "scaling",
              "vs_baseline", "dtype", "data", "config", "clocks", "e2e", "gpu_launches", "roofline", "cpu_baseline", "cut")
FINAL_MAX_BYTES = 4096


def _round(x, sig=5):
    if isinstance(x, float):
        return float(f"{x:.{sig}g}") if x == x and abs(x) != float("inf") else None
    if isinstance(x, dict):
        return {k: _round(v, sig) for k, v in x.items()}
    if isinstance(x, (list, tuple)):
        return [_round(v, sig) for v in x]
    return x


def final_line(full):
    """The compact last line from the full result dict: the contract's keys, the four whole-step speed-ups of the HCC
    order and ms + roofline fraction per stage and batch."""
    out = {k: full.get(k) for k in FINAL_KEYS}
    sp = full.get("speedup_hcc") or {}
    out["speedup_hcc"] = {k: sp.get(k) for k in ("pair_incl_vs_nosort", "pair_incl_vs_twopoint", "all_incl_vs_nosort", "all_incl_vs_twopoint")}
    st = full.get("stages_roofline_hcc") or {}
    out["stages_roofline_hcc"] = {b: {stg: {"ms": v.get("ms"), "bound": v.get("bound"), "frac": v.get("frac")} for stg, v in d.items()}
                                  for b, d in st.items()}
    if full.get("strong_scaling"):          # N > 1 only: the strong-scaling leg beside the weak-scaling value
        out["strong_scaling"] = {k: v for k, v in full["strong_scaling"].items() if k != "how"}
    line = json.dumps(_round(out), separators=(",", ":"))
    if len(line) >= FINAL_MAX_BYTES:       # never let a long free-text field cost the round its measurement
        for k in ("how", "traffic_unit", "peak_source", "sample", "parallelism"):
            for d in (out.get("e2e"), out.get("roofline"), out.get("cpu_baseline"), out.get("config")):
                if isinstance(d, dict) and k in d and isinstance(d[k], str):
                    d[k] = d[k][:60]
        line = json.dumps(_round(out), separators=(",", ":"))
    assert len(line) < FINAL_MAX_BYTES, len(line)
    return line


class ClockSampler:
    """nvidia-smi clocks and throttle reasons during the timed region (B200_PROFILING.md)."""
    Q = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,"
         "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,"
         "clocks_event_reasons.sw_power_cap")

    def __init__(self, index):
        self.index, self.rows, self.proc, self.thread = index, [], None, None

    def start(self):
        try:
            self.proc = subprocess.Popen(["nvidia-smi", "-i", str(self.index), f"--query-gpu={self.Q}",
                                          "--format=csv,noheader,nounits", "-lms", "20"],
                                         stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
        except Exception:
            self.proc = None
            return
        self.thread = threading.Thread(target=self._read, daemon=True)
        self.thread.start()

    def _read(self):
        for line in self.proc.stdout:
            self.rows.append((time.time(), line.strip()))

    def stop(self, t0, t1):
        if self.proc is None:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        time.sleep(0.15)
        self.proc.terminate()
        sm, smax, reasons = [], None, set()
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        for ts, line in self.rows:
            f = [x.strip() for x in line.split(",")]
            if len(f) < 7:
                continue
            try:
                c, m = float(f[0]), float(f[1])
            except ValueError:
                continue
            smax = m
            if t0 - 0.05 <= ts <= t1 + 0.15:
                sm.append(c)
                for nm, v in zip(names, f[3:7]):
                    if v.lower().startswith("active"):
                        reasons.add(nm)
        if not sm:   # region shorter than a sample period: take whatever was seen
            for ts, line in self.rows:
                f = [x.strip() for x in line.split(",")]
                try:
                    sm.append(float(f[0]))
                except Exception:
                    pass
        return {"sm_mhz": float(np.median(sm)) if sm else None, "sm_max_mhz": smax,
                "reasons": sorted(reasons), "samples": len(sm)}


# ------------------------------------------------------------------------------------------
def _oracle_tracer():
    import oracle

    def trace_closest(bvh, rays):
        t, p, _, _ = oracle.closest_bvh(rays, bvh.nodes, bvh.prim_idx, bvh.tris)
        return t, p
    return trace_closest


def oracle_pass(w, diffuse, shadow):
    """One pass of the hot path in the oracle: encode + stable sort + BVH traversal of both
    batches.  Returns seconds per stage."""
    import oracle
    b = w.bvh
    tables, _, _ = oracle.select_cut(b.nodes, w.K, w.key_bits)
    out = {"encode": 0.0, "sort": 0.0, "trace": 0.0}
    for rays, closest in ((diffuse, True), (shadow, False)):
        t0 = time.perf_counter()
        keys = oracle.encode_hcc(rays, b.nodes, tables)
        t1 = time.perf_counter()
        perm = oracle.sort(keys)
        t2 = time.perf_counter()
        r = np.ascontiguousarray(rays[perm])    # "fetches the rays based on these sorted indices"
        if closest:
            oracle.closest_bvh(r, b.nodes, b.prim_idx, b.tris)
        else:
            oracle.any_bvh(r, b.nodes, b.prim_idx, b.tris)
        t3 = time.perf_counter()
        out["encode"] += t1 - t0; out["sort"] += t2 - t1; out["trace"] += t3 - t2
    return out


def run_reference(args):
    """--impl reference: the CPU oracle as it stands, single-threaded, on a bounded sample."""
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return 0
    import hcc_inputs
    w = hcc_inputs.Workload(args.workload)
    n_d = min(args.ref_sample, w.width * w.height * w.spp)
    prim = w.primaries()[:n_d]
    t, p = _oracle_tracer()(w.bvh, prim)
    diffuse, shadow, _ = w.bounce(1, prim, t, p)
    n = diffuse.shape[0] + shadow.shape[0]
    for _ in range(args.warmup):
        oracle_pass(w, diffuse, shadow)
    t0 = time.perf_counter()
    split = {"encode": 0.0, "sort": 0.0, "trace": 0.0}
    for _ in range(args.steps):
        s = oracle_pass(w, diffuse, shadow)
        for k in split:
            split[k] += s[k]
    dt = time.perf_counter() - t0
    val = n * args.steps / dt / 1e6
    sample = (f"first {diffuse.shape[0]} diffuse + {shadow.shape[0]} shadow rays of the bounce "
              f"(primary-sample order) per step")
    line = {"impl": "reference", "metric": METRIC, "value": val, "unit": UNIT, "n_gpus": args.gpus,
            "steps": args.steps, "warmup": args.warmup, "ms_per_step": dt / args.steps * 1e3,
            "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f32",
            "data": "synthetic", "config": _config(args, w, diffuse.shape[0], shadow.shape[0], l2="n/a (CPU)"),
            "cpu_baseline": {"value": val, "unit": UNIT, "cores": 1, "kind": "oracle", "sample": sample,
                             "split_s": {k: v / args.steps for k, v in split.items()}, "host_cores": os.cpu_count()},
            "e2e": {"value": val, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
            "gpu_launches": 0}
    print(json.dumps(line))
    return 0


def _config(args, w, n_d, n_s, l2, workload=None, world=None):
    names = {"room": "config 2 'room' of BASELINE.json", "fig1": "config 3 'Figure-1-like' of BASELINE.json",
             "large": "config 5 'large' of BASELINE.json", "tiny": "config 1 'tiny' of BASELINE.json"}
    g = args.gpus if world is None else world
    return {"workload": names[workload or args.workload],
            "triangles": int(w.bvh.n_tris), "bvh_nodes": int(w.bvh.n_nodes), "K": int(w.K),
            "key_bits": int(w.key_bits), "diffuse_rays": int(n_d), "shadow_rays": int(n_s),
            "resolution": f"{w.width}x{w.height}x{w.spp}spp", "bounce": int(getattr(args, "bounce", 1)), "l2": l2,
            "parallelism": (f"{g} rank(s), one per GPU: every rank runs the whole path on its own batches (weak scaling); BVH and "
                            f"cut replicated, no collective on the data path; strong_scaling = one batch cut into contiguous ray ranges")}


# ------------------------------------------------------------------------------------------
class Scene:
    """One workload on the device: BVH, cut, the two ray batches of one bounce, scratch."""
    pass


def run_ours(args):
    import torch
    import torch.distributed as dist
    import hcc_inputs
    from paper_2305_16652_b200 import build as cuda_build
    cuda_build.build()
    import paper_2305_16652_b200 as hcc
    from paper_2305_16652_b200 import shard

    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if not torch.cuda.is_available():
        raise SystemExit("bench.py needs a CUDA device: the product path has no CPU fallback")
    # HCC_BENCH_SHARED_GPU=1 (code-path check on a one-GPU box, never a measurement): the ranks share the GPUs there are and
    # talk over gloo; no rank's kernels wait on another's, the collectives are the barrier, two reductions and one gather
    shared_gpu = os.environ.get("HCC_BENCH_SHARED_GPU") == "1"
    if shared_gpu:
        local %= torch.cuda.device_count()
    torch.cuda.set_device(local)
    if world > 1:
        if shared_gpu:
            dist.init_process_group("gloo")
        else:
            dist.init_process_group("nccl", device_id=torch.device("cuda", local))
    hbm_gbs, sm_max_mhz, peak_kind = _peaks()
    alu_peak = SM_COUNT * LANES_PER_SM * sm_max_mhz * 1e6 / 1e12     # T lane-op/s
    ev = lambda: torch.cuda.Event(enable_timing=True)
    flush = torch.empty(256 * 1024 * 1024 // 4, dtype=torch.int32, device="cuda")   # 256 MiB > 126 MB L2

    def max_over_ranks(x):
        if world == 1:
            return float(x)
        t = torch.tensor([x], dtype=torch.float64, device="cpu" if shared_gpu else "cuda")
        dist.all_reduce(t, op=dist.ReduceOp.MAX)
        return float(t.item())

    # ---- one workload on the device (seeded; rank r draws its own sub-pixel samples of the same scene)
    def load(name, res_scale=1.0, seed_rank=0):
        sc = Scene()
        sc.name = name
        sc.w = hcc_inputs.Workload(name, rank=seed_rank, res_scale=res_scale)
        b = sc.w.bvh
        sc.bvh = hcc.Bvh(b.nodes, b.tris, b.prim_idx)

        def gpu_trace_closest(_bvh, rays):
            h = hcc.trace(sc.bvh, torch.from_numpy(rays).cuda(), None, hcc.TRACE_CLOSEST)
            t, p, _, _ = hcc.hits_to_numpy(h)
            return t, p
        sc.trace_closest = gpu_trace_closest
        sc.had = hcc.density(sc.bvh)
        sc.cut = hcc.select_cut(sc.bvh, sc.had, sc.w.K, sc.w.key_bits)
        torch.cuda.synchronize()
        e0, e1 = ev(), ev()
        e0.record()
        hcc.density(sc.bvh, out=sc.had)
        hcc.select_cut(sc.bvh, sc.had, sc.w.K, sc.w.key_bits, cut=sc.cut)
        e1.record()
        torch.cuda.synchronize()
        sc.cut_ms = e0.elapsed_time(e1)
        sc.info = sc.cut.info()
        sc.bounce_no, sc.host = 0, None
        return sc

    def set_bounce(sc, bounce, shuffle=False):
        """Put the diffuse + shadow batches of `bounce` on the device (later bounces: trace the previous diffuse
        batch with the library's own tracer, spawn the next).  shuffle: the same rays in a seeded random order."""
        if sc.host is None or bounce < sc.bounce_no:
            sc.host, sc.bounce_no = sc.w.first_bounce(sc.trace_closest), 1
        while sc.bounce_no < bounce:
            t_prev, p_prev = sc.trace_closest(None, sc.host[0])
            d, s_, _ = sc.w.bounce(sc.bounce_no + 1, sc.host[0], t_prev, p_prev)
            sc.host, sc.bounce_no = (d, s_), sc.bounce_no + 1
        d_h, s_h = sc.host
        sc.n_d, sc.n_s = d_h.shape[0], s_h.shape[0]
        sc.n = sc.n_d + sc.n_s
        diffuse, shadow = torch.from_numpy(d_h).cuda(), torch.from_numpy(s_h).cuda()
        if shuffle:
            g = torch.Generator(device="cuda").manual_seed(0x5EED)
            diffuse = diffuse[torch.randperm(sc.n_d, device="cuda", generator=g)].contiguous()
            shadow = shadow[torch.randperm(sc.n_s, device="cuda", generator=g)].contiguous()
        sc.batches = ((diffuse, hcc.TRACE_CLOSEST, "diffuse"), (shadow, hcc.TRACE_ANY, "shadow"))
        if getattr(sc, "pipe", None) is None or sc.pipe.n_max < max(sc.n_d, sc.n_s):
            sc.pipe = hcc.Pipeline(max(sc.n_d, sc.n_s), 64, pair=True)
        sc.hits = {"diffuse": torch.empty((sc.n_d, 4), dtype=torch.float32, device="cuda"),
                   "shadow": torch.empty(sc.n_s, dtype=torch.uint8, device="cuda")}

    def step(sc, order):
        """One step = both batches of the bounce through the hot path, ONE C-ABI call (hcc_reorder_trace_pair)."""
        (ra, ma, na), (rb, mb, nb_) = sc.batches
        sc.pipe.reorder_trace_pair(sc.bvh, sc.cut, order, ra, ma, sc.hits[na], rb, mb, sc.hits[nb_], key_bits=sc.w.key_bits)

    def timed(sc, order, steps, warmup, per_stage=False):
        for _ in range(warmup):
            step(sc, order)
        torch.cuda.synchronize()
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()
        pairs = [(ev(), ev()) for _ in range(steps)]
        stage = {nm: {"encode": 0.0, "sort": 0.0, "trace": 0.0} for _, _, nm in sc.batches}
        t0 = time.time()
        for s_, e_ in pairs:
            flush.zero_()                       # L2 flush, outside the event bracket
            s_.record()
            if per_stage:
                sc.pipe.set_timing(True)
                for rays, mode, name in sc.batches:
                    sc.pipe.reorder_trace(sc.bvh, sc.cut, order, rays, mode, hits=sc.hits[name], key_bits=sc.w.key_bits)
                    ms = sc.pipe.stage_ms()
                    for k in stage[name]:
                        stage[name][k] += ms[k] / steps
                sc.pipe.set_timing(False)
            else:
                step(sc, order)
            e_.record()
        torch.cuda.synchronize()
        t1 = time.time()
        if world > 1:
            dist.barrier()
        ms = max_over_ranks(sum(s_.elapsed_time(e_) for s_, e_ in pairs))
        return ms / steps, stage, (t0, t1)

    ORDERS = (("hcc", hcc.ORDER_HCC), ("twopoint", hcc.ORDER_TWOPOINT), ("nosort", hcc.ORDER_NOSORT))

    def compare(sc, k):
        """Stage split of the three orders on the scene's current batches, and HCC's speed-ups."""
        orders = {}
        for name, order in ORDERS:
            ms, stage, _ = timed(sc, order, k, 3, per_stage=True)
            ms_pair, _, _ = timed(sc, order, k, 3)       # the same step as ONE hcc_reorder_trace_pair call (chained launches)
            o = {"ms_per_step": ms, "mrays_per_s_incl": sc.n / ms / 1e3, "pair_ms_per_step": ms_pair,
                 "pair_mrays_per_s_incl": sc.n / ms_pair / 1e3}
            for bn, nb in (("diffuse", sc.n_d), ("shadow", sc.n_s)):
                st = stage[bn]
                tot = st["encode"] + st["sort"] + st["trace"]
                o[bn] = {"encode_ms": st["encode"], "sort_ms": st["sort"], "trace_ms": st["trace"],
                         "mrays_per_s_incl": nb / tot / 1e3, "mrays_per_s_trace_only": nb / st["trace"] / 1e3}
            orders[name] = o
        speed = {}
        for bn in ("diffuse", "shadow"):
            h = orders["hcc"][bn]
            speed[bn] = {"incl_vs_nosort": h["mrays_per_s_incl"] / orders["nosort"][bn]["mrays_per_s_incl"],
                         "incl_vs_twopoint": h["mrays_per_s_incl"] / orders["twopoint"][bn]["mrays_per_s_incl"],
                         "trace_vs_nosort": h["mrays_per_s_trace_only"] / orders["nosort"][bn]["mrays_per_s_trace_only"],
                         "trace_vs_twopoint": h["mrays_per_s_trace_only"] / orders["twopoint"][bn]["mrays_per_s_trace_only"]}
        speed["all_incl_vs_nosort"] = orders["nosort"]["ms_per_step"] / orders["hcc"]["ms_per_step"]
        speed["all_incl_vs_twopoint"] = orders["twopoint"]["ms_per_step"] / orders["hcc"]["ms_per_step"]
        speed["pair_incl_vs_nosort"] = orders["nosort"]["pair_ms_per_step"] / orders["hcc"]["pair_ms_per_step"]
        speed["pair_incl_vs_twopoint"] = orders["twopoint"]["pair_ms_per_step"] / orders["hcc"]["pair_ms_per_step"]
        return orders, speed

    def order_perms(sc, rays):
        """The three traced orders of one batch as permutations (None = NoSort) and the HCC keys."""
        keys = hcc.encode(rays, sc.cut)
        keys0 = keys.clone()
        perm = hcc.sort(keys, sc.info["bits_used"])
        tk = hcc.encode_twopoint(rays, sc.bvh.scene_lo, sc.bvh.scene_hi, sc.w.key_bits)
        perm_t = hcc.sort(tk, 6 * (sc.w.key_bits // 6))
        return {"nosort": None, "twopoint": perm_t, "hcc": perm}, keys0

    def counters(sc):
        """What a warp shares: work counters of the instrumented traversal kernel (never timed) for the three orders
        (coherent rays fetch the same nodes) and ANC."""
        out = {}
        for rays, mode, name in sc.batches:
            perms, keys0 = order_perms(sc, rays)
            o = {}
            for on, pm in perms.items():
                st = hcc.trace_stats(sc.bvh, rays, pm, mode)
                o[on] = {"node_records_per_ray": st["nodes"] / max(st["rays"], 1), "tri_tests_per_ray": st["tris"] / max(st["rays"], 1),
                         "distinct_records_per_warp_step": st["records_per_step"], "lanes_per_warp_step": st["lanes_per_step"],
                         "tri_tests_per_round": st["tri_tests_per_round"], "max_stack": st["max_stack"],
                         "lane_ops": st["nodes"] * OPS_NODE + st["tris"] * OPS_TRI,
                         "lane_cycles": st["nodes"] * CYC_NODE + st["tris"] * CYC_TRI}
            out[name] = {"anc_hcc": hcc.anc(keys0, perms["hcc"]), "anc_nosort": hcc.anc(keys0, None), "orders": o}
        return out

    # =========================================================================== the headline workload
    sc = load(args.workload, args.res_scale, seed_rank=rank)
    set_bounce(sc, args.bounce)
    w, bvh, cut, info = sc.w, sc.bvh, sc.cut, sc.info
    n_d, n_s, n = sc.n_d, sc.n_s, sc.n
    container = info["container_bits"]
    passes = (info["bits_used"] + 7) // 8
    pipe, hits_d, hits_s = sc.pipe, sc.hits["diffuse"], sc.hits["shadow"]
    (diffuse, _, _), (shadow, _, _) = sc.batches
    diffuse_h, shadow_h = sc.host

    # ---- the timed region: K steps of the HCC-ordered hot path
    sampler = ClockSampler(local)
    if rank == 0:
        sampler.start()
        time.sleep(0.3)
    ms_step, _, (t0, t1) = timed(sc, hcc.ORDER_HCC, args.steps, args.warmup)
    clocks = sampler.stop(t0, t1) if rank == 0 else None
    value = world * n / (ms_step * 1e-3) / 1e6

    # ---- stage split and the comparison orders on the same rays (short runs, same hygiene)
    k_cmp = max(3, min(args.steps, 20))
    orders, speed = compare(sc, k_cmp)

    # ---- PAPER.md:428's sort-cost reduction on the same step: only the first level's field of the code is sorted (the
    #      lower levels' bits are left unordered); reported beside `value`, which keeps the full sort
    skip = info["bits_used"] - info["widths"][0] if len(info["widths"]) > 1 else 0
    sc.pipe.set_sort_skip_bits(skip)
    ms_trunc, _, _ = timed(sc, hcc.ORDER_HCC, k_cmp, 3)
    sc.pipe.set_sort_skip_bits(0)
    truncated = {"skip_bits": skip, "sorted_bits": info["bits_used"] - skip, "ms_per_step": ms_trunc, "value": world * n / ms_trunc / 1e3,
                 "unit": UNIT, "how": "hcc_pipeline_set_sort_skip_bits: the sort orders the first level's field only (PAPER.md:428)"}

    # ---- the same step with the two batches of the bounce on two streams (one pipeline each)
    pipe2 = hcc.Pipeline(n_d, 64)
    streams_o = (torch.cuda.Stream(), torch.cuda.Stream())

    def step_overlapped():
        cur = torch.cuda.current_stream()
        for st in streams_o:
            st.wait_stream(cur)
        pipe.reorder_trace(bvh, cut, hcc.ORDER_HCC, shadow, hcc.TRACE_ANY, hits=hits_s, key_bits=w.key_bits, stream=streams_o[0])
        pipe2.reorder_trace(bvh, cut, hcc.ORDER_HCC, diffuse, hcc.TRACE_CLOSEST, hits=hits_d, key_bits=w.key_bits, stream=streams_o[1])
        for st in streams_o:
            cur.wait_stream(st)
    for _ in range(3):
        step_overlapped()
    torch.cuda.synchronize()
    ov = []
    for _ in range(k_cmp):
        flush.zero_()
        s0, e0 = ev(), ev()
        s0.record(); step_overlapped(); e0.record()
        torch.cuda.synchronize()
        ov.append(s0.elapsed_time(e0))
    ov_ms = max_over_ranks(float(np.mean(ov)))
    overlapped = {"ms_per_step": ov_ms, "value": world * n / ov_ms / 1e3, "unit": UNIT,
                  "how": "diffuse and shadow batch of the step on two streams, one hcc_pipeline each"}
    del pipe2

    # ---- strong scaling over the ranks: ONE batch pair (rank 0's samples) cut into contiguous ray ranges
    #      (shard.ray_shard), every rank running hcc_reorder_trace on its range; no collective on the data path,
    #      the hits are gathered once afterwards
    strong = None
    if world > 1:
        sc0 = sc if rank == 0 else load(args.workload, args.res_scale, seed_rank=0)
        if sc0 is not sc:
            set_bounce(sc0, args.bounce)
        shard_len = lambda n_: shard.ray_shard(n_, 0, world)[1] - shard.ray_shard(n_, 0, world)[0]
        spipe = hcc.Pipeline(max(shard_len(sc0.n_d), shard_len(sc0.n_s), 1), 64)

        def sstep():
            return [shard.sharded_reorder_trace(spipe, sc0.bvh, sc0.cut, hcc.ORDER_HCC, rays, mode, rank, world,
                                                key_bits=sc0.w.key_bits)[0] for rays, mode, _ in sc0.batches]
        for _ in range(3):
            sstep()
        torch.cuda.synchronize()
        dist.barrier()
        tot = 0.0
        for _ in range(k_cmp):
            flush.zero_()
            s0, e0 = ev(), ev()
            s0.record(); loc = sstep(); e0.record()
            torch.cuda.synchronize()
            tot += s0.elapsed_time(e0) / k_cmp
        dist.barrier()
        s_ms = max_over_ranks(tot)
        full_d = shard.gather_hits(loc[0], sc0.n_d)     # once, for the consumer; not part of the path
        full_s = shard.gather_hits(loc[1], sc0.n_s)
        ok = True
        if rank == 0:
            ok = bool(torch.equal(full_d.view(torch.int32), hcc.trace(sc0.bvh, sc0.batches[0][0], None, hcc.TRACE_CLOSEST).view(torch.int32))
                      and torch.equal(full_s, hcc.trace(sc0.bvh, sc0.batches[1][0], None, hcc.TRACE_ANY)))
        strong = {"ms_per_step": s_ms, "value": sc0.n / s_ms / 1e3, "unit": UNIT, "scaling": "strong", "ranks": world,
                  "rays_total": sc0.n, "gathered_hits_equal_unsharded": ok,
                  "how": "one bounce's batches cut into contiguous ray ranges by shard.ray_shard, one range per rank"}

    # ---- trace work counters for the three orders (instrumented kernel, never timed) and ANC
    diag = counters(sc)
    nrays = {"diffuse": n_d, "shadow": n_s}
    key_b = container // 8
    sb_algo, sb_real = sort_bytes(key_b, passes)
    stages = {}
    for name in ("diffuse", "shadow"):
        o, nb = orders["hcc"][name], nrays[name]
        enc_gbs = nb * (32 + key_b) / (o["encode_ms"] * 1e-3) / 1e9
        sort_gbs = nb * sb_real / (o["sort_ms"] * 1e-3) / 1e9
        tr = diag[name]["orders"]["hcc"]["lane_ops"] / (o["trace_ms"] * 1e-3) / 1e12
        enc_ops = nb * info["bits_used"] * OPS_BOX / (o["encode_ms"] * 1e-3) / 1e12
        stages[name] = {
            "encode": {"ms": o["encode_ms"], "bound": "hbm", "achieved": enc_gbs, "peak": hbm_gbs, "unit": "GB/s", "frac": enc_gbs / hbm_gbs,
                       "alu_achieved_tlaneops": enc_ops, "alu_frac": enc_ops / alu_peak, "box_tests_per_ray": info["bits_used"],
                       # the same fraction with the op counts of SURVEY.md:604 (20 per test; 14 with 3-input min/max) beside the definition's 26
                       "alu_frac_by_ops_per_test": {str(k_): enc_ops * k_ / OPS_BOX / alu_peak for k_ in (OPS_BOX, 20, 14)}},
            "sort": {"ms": o["sort_ms"], "bound": "hbm", "achieved": sort_gbs, "peak": hbm_gbs, "unit": "GB/s", "frac": sort_gbs / hbm_gbs,
                     "passes": passes, "bytes_per_pair_moved": sb_real, "bytes_per_pair_survey": sb_algo,
                     "frac_survey_bytes": nb * sb_algo / (o["sort_ms"] * 1e-3) / 1e9 / hbm_gbs},
            "trace": {"ms": o["trace_ms"], "bound": "alu", "achieved": tr, "peak": alu_peak, "unit": "Tlaneop/s", "frac": tr / alu_peak,
                      "frac_pipe_weighted": diag[name]["orders"]["hcc"]["lane_cycles"] / (o["trace_ms"] * 1e-3) / 1e12 / alu_peak}}
    # dominant kernel of the step
    dom = max((("diffuse", "trace"), ("shadow", "trace"), ("diffuse", "sort"), ("shadow", "sort"),
               ("diffuse", "encode"), ("shadow", "encode")), key=lambda k: orders["hcc"][k[0]][k[1] + "_ms"])
    roof = dict(stages[dom[0]][dom[1]])
    plain = dom[1] == "trace" and args.bounce == 1 and args.res_scale == 1.0 and world == 1
    roof = {"bound": roof["bound"], "achieved": roof["achieved"], "peak": roof["peak"], "unit": roof["unit"],
            "frac": roof["frac"],
            "traffic": ncu_traffic(args.workload, dom[0]) if plain else None,
            "traffic_unit": "bytes per launch (dram read + write, ncu --set full; profiles/r3_trace_traffic.md, null when the "
                            "kernel sources changed since the capture)",
            "kernel": f"{dom[1]} ({dom[0]} batch)",
            "peak_source": (f"{peak_kind} HBM copy" if roof["bound"] == "hbm" else
                            f"148 SMs x 128 fp32 lanes x {sm_max_mhz:.0f} MHz (DESIGN.md)")}

    # ---- later bounces and shuffled input of the headline scene: the regimes in which the rays are NOT already in
    #      camera order (PAPER.md:294-299 measures secondary rays of every bounce)
    by_bounce = {str(args.bounce): {"speedup_hcc": speed, "rays": n,
                                    "trace_ms": {o: {b_: orders[o][b_]["trace_ms"] for b_ in ("diffuse", "shadow")} for o in orders}}}
    shuffled = None
    def warp_counters(sc_):
        """Per batch and order: distinct node records and lanes per warp-level node step, node records per ray (hcc_trace_stats)."""
        return {bn: {on: {k_: v_[k_] for k_ in ("distinct_records_per_warp_step", "lanes_per_warp_step", "node_records_per_ray", "tri_tests_per_ray")}
                     for on, v_ in d_["orders"].items()} for bn, d_ in counters(sc_).items()}

    def bounce_entry(sc_, o_b, s_b):
        return {"speedup_hcc": s_b, "rays": sc_.n, "rays_diffuse": sc_.n_d, "rays_shadow": sc_.n_s,
                "trace_ms": {o: {b_: o_b[o][b_]["trace_ms"] for b_ in ("diffuse", "shadow")} for o in o_b},
                "encode_sort_ms": {o: {b_: o_b[o][b_]["encode_ms"] + o_b[o][b_]["sort_ms"] for b_ in ("diffuse", "shadow")} for o in o_b},
                "incl_ms_per_step": {o: o_b[o]["ms_per_step"] for o in o_b},
                "pair_ms_per_step": {o: o_b[o]["pair_ms_per_step"] for o in o_b},
                "warp_counters": warp_counters(sc_)}

    if world == 1 and args.bounces > 0:
        by_bounce[str(args.bounce)] = bounce_entry(sc, orders, speed)
        k_b = max(3, min(args.steps, 10))
        for b_i in range(args.bounce + 1, args.bounce + 1 + args.bounces):
            set_bounce(sc, b_i)
            o_b, s_b = compare(sc, k_b)
            by_bounce[str(b_i)] = bounce_entry(sc, o_b, s_b)
        set_bounce(sc, args.bounce, shuffle=True)
        o_s, s_s = compare(sc, k_b)
        shuffled = {**bounce_entry(sc, o_s, s_s),
                    "how": "the same two batches in a seeded random order (a wavefront renderer does not emit rays in camera order)"}
        set_bounce(sc, args.bounce)
        step(sc, hcc.ORDER_HCC)      # the hit buffers hold the unshuffled batches' results again (checked by the e2e leg)
        hits_d, hits_s = sc.hits["diffuse"], sc.hits["shadow"]
        (diffuse, _, _), (shadow, _, _) = sc.batches

    # ---- encode and sort at the batch size of configs 3/5 (the shadow batch tiled to ~33.5 M rays): the
    #      config-2 batches (1-2 M pairs) are launch- and latency-bound, so the HBM fractions that the
    #      north_star's 60 % bar is about are measured here (SURVEY.md §7 "hard parts", §8(d))
    def med(fn, setup=None, k=7):
        out = []
        for i in range(k + 2):
            if setup:
                setup()
            flush.zero_()
            s0, e0 = ev(), ev()
            s0.record(); fn(); e0.record()
            torch.cuda.synchronize()
            if i >= 2:
                out.append(s0.elapsed_time(e0))
        return float(np.median(out))

    large = None
    if world == 1 and args.large_n:
        reps = max(1, (1 << 25) // n_s)
        big = shadow.repeat(reps, 1) if reps > 1 else shadow
        nb = big.shape[0]

        def hbm_leg(ms, nbytes, **extra):
            return {"ms": ms, "bound": "hbm", "achieved": nbytes / ms / 1e6, "peak": hbm_gbs, "unit": "GB/s",
                    "frac": nbytes / ms / 1e6 / hbm_gbs, **extra}

        def sort_leg(keys, bits_used, cb):
            keys0 = keys.clone()
            ws = torch.empty(hcc.sort_workspace_bytes(nb, cb), dtype=torch.uint8, device="cuda")
            pm = torch.empty(nb, dtype=torch.int32, device="cuda")
            ms = med(lambda: hcc.sort(keys, bits_used, perm=pm, workspace=ws), setup=lambda: keys.copy_(keys0))
            p_ = (bits_used + 7) // 8
            algo, real = sort_bytes(cb // 8, p_)
            return hbm_leg(ms, nb * real, passes=p_, bytes_per_pair_moved=real, bytes_per_pair_survey=algo,
                           frac_survey_bytes=nb * algo / ms / 1e6 / hbm_gbs)
        keys_b = hcc.encode(big, cut)
        enc_ms = med(lambda: hcc.encode(big, cut, keys=keys_b))
        tkb = 4 if w.key_bits <= 32 else 8
        tp_keys = hcc.encode_twopoint(big, bvh.scene_lo, bvh.scene_hi, w.key_bits)
        tp_ms = med(lambda: hcc.encode_twopoint(big, bvh.scene_lo, bvh.scene_hi, w.key_bits, keys=tp_keys))
        large = {"rays": int(nb), "how": f"shadow batch tiled x{reps}",
                 "encode": hbm_leg(enc_ms, nb * (32 + container // 8), box_tests_per_ray=info["bits_used"],
                                   alu_frac=nb * info["bits_used"] * OPS_BOX / (enc_ms * 1e-3) / 1e12 / alu_peak),
                 "sort": sort_leg(keys_b, info["bits_used"], container),
                 "encode_twopoint": hbm_leg(tp_ms, nb * (32 + tkb)),
                 "sort_twopoint_keys": sort_leg(tp_keys, 6 * (w.key_bits // 6), 32 if w.key_bits <= 32 else 64)}
        # the paper's own MLHCC16 (8 x 8 entries, 16 slab tests per ray): SURVEY.md 8(d) expects
        # codes of <= 16 tests to be HBM-bound
        cut16 = hcc.select_cut_levels(bvh, sc.had, [8, 8], 16)
        keys16 = hcc.encode(big, cut16)
        e16 = med(lambda: hcc.encode(big, cut16, keys=keys16))
        large["encode_mlhcc16"] = hbm_leg(e16, nb * (32 + 4), box_tests_per_ray=16,
                                          alu_frac=nb * 16 * OPS_BOX / (e16 * 1e-3) / 1e12 / alu_peak)
        del big, keys_b, tp_keys, keys16
        torch.cuda.empty_cache()

    # ---- the other single-GPU configs of BASELINE.json at their stated sizes: one bounce of config 3 ("fig1") and
    #      of config 5 ("large"), three orders each
    others = None
    if world == 1 and args.configs:
        others = {}
        for name in args.configs.split(","):
            if name == args.workload:
                continue
            t_load = time.time()
            so = load(name, 1.0)
            set_bounce(so, 1)
            t_load = time.time() - t_load
            k_o = 3
            ms_o, _, _ = timed(so, hcc.ORDER_HCC, k_o, 3)
            o_o, s_o = compare(so, k_o)
            sb = sort_bytes(so.info["container_bits"] // 8, (so.info["bits_used"] + 7) // 8)
            others[name] = {"config": _config(args, so.w, so.n_d, so.n_s, l2="flushed between timed steps", workload=name),
                            "value": so.n / ms_o / 1e3, "unit": UNIT, "ms_per_step": ms_o, "steps": k_o,
                            "cut": {"widths": so.info["widths"], "bits_used": so.info["bits_used"], "cut_ms": so.cut_ms},
                            "orders": o_o, "speedup_hcc": s_o,
                            "sort_frac_of_hbm": {b_: nb_ * sb[1] / (o_o["hcc"][b_]["sort_ms"] * 1e-3) / 1e9 / hbm_gbs
                                                 for b_, nb_ in (("diffuse", so.n_d), ("shadow", so.n_s))},
                            "encode_frac_of_hbm": {b_: nb_ * (32 + so.info["container_bits"] // 8) / (o_o["hcc"][b_]["encode_ms"] * 1e-3) / 1e9 / hbm_gbs
                                                   for b_, nb_ in (("diffuse", so.n_d), ("shadow", so.n_s))},
                            "counters": counters(so) if args.counters_all else None,
                            "input_generation_s": t_load}
            del so
            torch.cuda.empty_cache()

    # ---- studies, on request: f1 sort truncation, f2 lambda and
    #      ANC, f3 prefix path code (:116-128), f4 regular grid (:243)
    studies = None
    if args.studies and world == 1:
        batches = sc.batches
        hits = sc.hits
        had = sc.had

        def med_ms(fn, setup=None, k=5):
            return med(fn, setup, k)

        def run_order(make_keys, bits_used, bit_lo=0):
            """encode / sort / trace medians and ANC per batch for one key function (None = NoSort)."""
            res = {}
            for rays, mode, name in batches:
                nb = rays.shape[0]
                if make_keys is None:
                    tr = med_ms(lambda: hcc.trace(bvh, rays, None, mode, hits=hits[name]))
                    res[name] = {"encode_ms": 0.0, "sort_ms": 0.0, "trace_ms": tr, "mrays_per_s_incl": nb / tr / 1e3,
                                 "mrays_per_s_trace_only": nb / tr / 1e3}
                    continue
                keys = make_keys(rays)
                keys0 = keys.clone()
                cb = 32 if keys.dtype == torch.int32 else 64
                ws = torch.empty(hcc.sort_workspace_bytes(nb, cb), dtype=torch.uint8, device="cuda")
                perm = torch.empty(nb, dtype=torch.int32, device="cuda")
                enc = med_ms(lambda: make_keys(rays, keys))
                srt = med_ms(lambda: hcc.sort(keys, bits_used, perm=perm, workspace=ws, bit_lo=bit_lo), setup=lambda: keys.copy_(keys0))
                tr = med_ms(lambda: hcc.trace(bvh, rays, perm, mode, hits=hits[name]))
                res[name] = {"encode_ms": enc, "sort_ms": srt, "trace_ms": tr, "mrays_per_s_incl": nb / (enc + srt + tr) / 1e3,
                             "mrays_per_s_trace_only": nb / tr / 1e3, "anc": hcc.anc(keys0, perm)}
            return res

        hcc_keys = lambda cut_: (lambda rays, keys=None: hcc.encode(rays, cut_, keys=keys))
        studies = {"truncation": {}, "lambda": {}, "orders": {}}
        for skip in (0, 8, 16, 24, info["bits_used"]):
            if skip <= info["bits_used"]:
                studies["truncation"][f"skip_{skip}_bits"] = run_order(hcc_keys(cut), info["bits_used"], bit_lo=skip)
        for lam in (0.1, 0.125, 0.25, 0.5, 1.0):
            cut_l = hcc.select_cut(bvh, hcc.density(bvh, lam), w.K, w.key_bits)
            studies["lambda"][f"{lam}"] = run_order(hcc_keys(cut_l), cut_l.info()["bits_used"])
        grid_cut = hcc.select_grid(bvh, info["widths"], w.key_bits)
        tp_bits = 6 * (w.key_bits // 6)
        studies["orders"] = {
            "nosort": run_order(None, 0),
            "twopoint": run_order(lambda rays, keys=None: hcc.encode_twopoint(rays, bvh.scene_lo, bvh.scene_hi, w.key_bits, keys=keys), tp_bits),
            "hcc": run_order(hcc_keys(cut), info["bits_used"]),
            "grid": run_order(hcc_keys(grid_cut), info["bits_used"]),
            "ppc": run_order(lambda rays, keys=None: hcc.encode_ppc(bvh, rays, w.key_bits, keys=keys), w.key_bits)}
        if len(info["widths"]) > 1:      # Algorithm 3 as printed (small popped nodes dropped) instead of reading R4
            lit_cut = hcc.select_cut_levels(bvh, had, info["widths"], w.key_bits, flags=hcc.CUT_ALG3_DISCARD)
            studies["orders"]["hcc_alg3_discard"] = run_order(hcc_keys(lit_cut), info["bits_used"])
        # config 4 of BASELINE.json: cut size x key length on the same rays (Tables 6-7 analogue)
        sweep = []
        for kb in (16, 24, 32, 48, 64):
            tp = run_order(lambda rays, keys=None, kb=kb: hcc.encode_twopoint(rays, bvh.scene_lo, bvh.scene_hi, kb, keys=keys), 6 * (kb // 6))
            sweep.append({"order": "twopoint", "key_bits": kb, "bits_used": 6 * (kb // 6), **tp})
            for K in (256, 1024, 4096, 16384, 65536):
                cut_s = hcc.select_cut(bvh, had, K, kb)
                i_s = cut_s.info()
                if any(e["order"] == "hcc" and e["key_bits"] == kb and e["widths"] == i_s["widths"] for e in sweep):
                    continue      # capped to a hierarchy already measured at this key length
                sweep.append({"order": "hcc", "key_bits": kb, "K": K, "K_eff": i_s["K_eff"], "widths": i_s["widths"],
                              "bits_used": i_s["bits_used"], **run_order(hcc_keys(cut_s), i_s["bits_used"])})
        studies["sweep"] = sweep
        step(sc, hcc.ORDER_HCC)
        studies["note"] = ("per batch medians of 5; grid = regular-grid tables of the same widths through the same encoder; "
                           "ppc = prefix path code with key_bits tests (upper-bound ordering, PAPER.md:128)")

    # ---- e2e: the same step through the C ABI with HOST buffers (pinned), copies inside the timing
    rays_pin = {"diffuse": torch.from_numpy(diffuse_h).pin_memory(), "shadow": torch.from_numpy(shadow_h).pin_memory()}
    hits_pin = {"diffuse": torch.empty((n_d, 4), dtype=torch.float32).pin_memory(),
                "shadow": torch.empty(n_s, dtype=torch.uint8).pin_memory()}

    # the batches are streamed in chunks of about half a million rays, each through a pipeline and a stream of its own
    # (hcc_reorder_trace_host_async: copy in, encode, sort, trace, copy out): the host->device copies queue up on the copy
    # engine back to back while the kernels of the chunks already on the device run, and hits go back as chunks finish.
    # A chunk is sorted within itself (coherence is made per chunk); hits do not depend on the order.
    e2e_chunk = max(1, args.e2e_chunk)
    chunks = []           # (name, mode, start, stop)
    for _, mode, name in sc.batches:
        nb = nrays[name]
        parts = max(1, (nb + e2e_chunk - 1) // e2e_chunk)
        for k in range(parts):
            a_, b_ = shard.ray_shard(nb, k, parts)
            chunks.append((name, mode, a_, b_))
    pipes_h = [hcc.Pipeline(max(b_ - a_, 1), 64, host_staging=True) for _, _, a_, b_ in chunks]
    streams_h = [torch.cuda.Stream() for _ in chunks]

    def step_host():
        cur = torch.cuda.current_stream()
        for (name, mode, a_, b_), ph, st in zip(chunks, pipes_h, streams_h):
            st.wait_stream(cur)
            ph.reorder_trace_host_async(bvh, cut, hcc.ORDER_HCC, rays_pin[name][a_:b_], hits_pin[name][a_:b_], mode,
                                        key_bits=w.key_bits, stream=st)
        for ph, st in zip(pipes_h, streams_h):
            ph.synchronize()
            cur.wait_stream(st)
    for _ in range(3):
        step_host()
    torch.cuda.synchronize()
    if world > 1:
        dist.barrier()
    k_e2e = max(3, min(args.steps, 10))
    e2e_ms = 0.0
    for _ in range(k_e2e):
        flush.zero_()
        s_, e_ = ev(), ev()
        s_.record()
        step_host()
        e_.record()
        torch.cuda.synchronize()
        e2e_ms += s_.elapsed_time(e_) / k_e2e
    e2e_ms = max_over_ranks(e2e_ms)
    step(sc, hcc.ORDER_HCC)
    assert torch.equal(hits_pin["shadow"].cuda(), hits_s) and torch.equal(hits_pin["diffuse"].cuda().view(torch.int32), hits_d.view(torch.int32))
    e2e = {"value": world * n / e2e_ms / 1e3, "unit": UNIT, "ms_per_step": e2e_ms,
           "h2d_bytes_per_step": 32 * n, "d2h_bytes_per_step": 16 * n_d + n_s,
           "how": f"{len(chunks)} chunks of <= {e2e_chunk} rays, one hcc_reorder_trace_host_async each on a stream of its own"}

    # kernels launched per step: per batch 1 key kernel + (init + histogram + scan + one per digit) + 1 trace
    launches_per_step = 2 * (1 + (3 + passes) + 1)

    if rank != 0:
        if world > 1:
            dist.destroy_process_group()
        return 0

    # ---- cpu_baseline: the oracle on this box's host cores, bounded sample, rank 0, N = 1 only
    cpu = None
    if world == 1 and not args.no_cpu_baseline:
        m_d = min(n_d, args.cpu_sample)
        d_s, s_s = diffuse_h[:m_d], shadow_h[:2 * m_d]
        t0 = time.perf_counter()
        split = oracle_pass(w, d_s, s_s)
        dt = time.perf_counter() - t0
        cpu = {"value": (d_s.shape[0] + s_s.shape[0]) / dt / 1e6, "unit": UNIT, "cores": 1, "kind": "oracle",
               "sample": f"first {d_s.shape[0]} diffuse + {s_s.shape[0]} shadow rays of the same batches, one pass "
                         f"(encode + stable sort + BVH traversal), {dt:.1f} s",
               "split_s": split, "host_cores": os.cpu_count()}

    line = {"metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps, "warmup": args.warmup,
            "ms_per_step": ms_step, "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f32",
            "data": "synthetic",
            "config": dict(_config(args, w, n_d, n_s, l2="flushed between timed steps (256 MiB write)", world=world),
                           lib=os.path.relpath(hcc.LIB_PATH, ROOT), no_pdl=os.environ.get("HCC_NO_PDL") == "1",
                           **({"shared_gpu_code_path_check": True} if shared_gpu else {})),
            "clocks": clocks, "e2e": e2e, "gpu_launches": launches_per_step * args.steps,
            "roofline": roof, "cpu_baseline": cpu,
            "cut": {"widths": info["widths"], "K_eff": info["K_eff"], "bits_used": info["bits_used"],
                    "container_bits": container, "cut_ms": sc.cut_ms},
            "orders": orders, "speedup_hcc": speed, "speedup_hcc_by_bounce": by_bounce, "shuffled_input": shuffled,
            "stages_roofline_hcc": stages, "stages_roofline_large_batch": large, "two_stream_step": overlapped, "sort_truncated_step": truncated,
            "strong_scaling": strong, "other_configs": others, "studies": studies,
            "diagnostics": diag,
            "paper_context": "RTX 3060, Breakfast: HCC 67.6 vs NoSort 37.4 vs TwoPoint 56.8 Mrays/s trace-only (PAPER.md:294-299); not comparable"}
    if args.full_json:
        with open(args.full_json, "w") as f:
            json.dump(line, f)
    # what the flags asked for beyond the headline: one JSON line per section, BEFORE the final line
    for name in ("orders", "speedup_hcc", "stages_roofline_hcc", "two_stream_step", "sort_truncated_step", "diagnostics",
                 "speedup_hcc_by_bounce", "shuffled_input", "stages_roofline_large_batch", "strong_scaling", "other_configs", "studies"):
        if args.sections and line.get(name) is not None:
            print(json.dumps({"section": name, "data": _round(line[name], 6)}, separators=(",", ":")))
    sys.stdout.flush()
    print(final_line(line))
    if world > 1:
        dist.destroy_process_group()
    return 0


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=100)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--workload", default="room", choices=["tiny", "room", "fig1", "large"])
    ap.add_argument("--cpu-sample", type=int, default=1 << 20, help="diffuse rays in the cpu_baseline sample")
    ap.add_argument("--ref-sample", type=int, default=1 << 15, help="diffuse rays per step of --impl reference")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--bounce", type=int, default=1, help="which bounce's ray batches to run (1 = rays off the primary hits)")
    ap.add_argument("--res-scale", type=float, default=1.0, help="image scale of the workload (1.0 = the config's resolution)")
    ap.add_argument("--studies", action="store_true",
                    help="the NEXT-row studies: sort truncation, lambda/ANC, grid and PPC orders, config-4 sweep (about 45 s; off by default)")
    ap.add_argument("--no-studies", dest="studies", action="store_false", help="(default)")
    ap.add_argument("--large-n", action="store_true", help="the large-batch (33.5 M rays) encode/sort roofline leg")
    ap.add_argument("--no-large-n", dest="large_n", action="store_false", help="(default)")
    ap.add_argument("--configs", default="", help="comma list of further configs to run at their stated sizes (fig1,large): other_configs")
    ap.add_argument("--bounces", type=int, default=0,
                    help="also run the three orders on this many LATER bounces of the workload and on its shuffled first batch (speedup_hcc_by_bounce, shuffled_input)")
    ap.add_argument("--full-json", default="", help="write the complete result (every section) to this file")
    ap.add_argument("--sections", action="store_true",
                    help="print every section of the result as its own JSON line before the final compact line")
    ap.add_argument("--counters-all", action="store_true", help="per-order trace counters for --configs too")
    ap.add_argument("--e2e-chunk", type=int, default=1 << 19, help="rays per chunk of the host-buffer (e2e) leg")
    ap.add_argument("--quick", action="store_true", help="(default; kept for old command lines) no later-bounce and shuffled-input legs")
    args = ap.parse_args()
    if args.warmup < 3 and args.impl == "ours":
        args.warmup = 3
    if args.gpus > 1 and "WORLD_SIZE" not in os.environ:
        # plain `python bench.py --gpus N`: start the N ranks ourselves (one process per GPU, NCCL)
        import socket
        with socket.socket() as sk:
            sk.bind(("127.0.0.1", 0))
            port = sk.getsockname()[1]
        cmd = [sys.executable, "-m", "torch.distributed.run", "--nnodes=1", f"--nproc-per-node={args.gpus}",
               "--master-addr", "127.0.0.1", "--master-port", str(port), os.path.abspath(__file__)] + sys.argv[1:]
        return subprocess.call(cmd)
    world_env = int(os.environ.get("WORLD_SIZE", "1"))
    if world_env != args.gpus:
        raise SystemExit(f"bench.py: --gpus {args.gpus} but WORLD_SIZE={world_env}: launch with --nproc-per-node {args.gpus}")
    return run_reference(args) if args.impl == "reference" else run_ours(args)


if __name__ == "__main__":
    sys.exit(main())
