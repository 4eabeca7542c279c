"""bench.py — the hot path of hierarchy-cut-code ray reordering on B200, measured.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--impl ours|reference] [--workload room|fig1|tiny]

One STEP = one pass of the whole per-batch hot path (Figure 11) over one
bounce of BASELINE.json config 2 ("room": 64,012 triangles, 512x512x4 spp): the diffuse batch
(1,048,576 closest-hit rays) and the shadow batch (2,097,152 any-hit rays), each
key-computed (hcc_encode), sorted (hcc_sort) and traced through the sorted indices (hcc_trace)
in ONE C-ABI call, hcc_reorder_trace.  Metric: secondary Mrays/s INCLUDING encode + sort.
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
#  trace : lane-operations = 34 per sibling-pair record (12 cell->float conversions, 12 fma, 8 min/max,
#          2 compares: both quantised child boxes, trace.cu) + 36 per triangle test (the formula in
#          include/hcc.h); encode: 26 per exact fp32 slab test (6 sub, 6 mul, 12 min/max, compare, bit).
OPS_BOX, OPS_NODE, OPS_TRI = 26, 68, 36
# dram__bytes_read.sum + dram__bytes_write.sum per launch of the two trace kernels on config 2, from the
# ncu --set full capture summarised in profiles/r1b_ncu_full.md (a profiler number, config "room" only)
NCU_TRAFFIC_ROOM = {"diffuse": 41.140480e6 + 0.928000e6, "shadow": 79.290880e6 + 5.325568e6}
SM_COUNT, LANES_PER_SM = 148, 128


def _peaks():
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    try:
        with open(p) as f:
            d = json.load(f)
        return float(d["hbm_gbs"]), float(d.get("sm_max_mhz", 1965.0)), "measured"
    except Exception:
        return 6650.0, 1965.0, "fallback"


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


def _config(args, w, n_d, n_s, l2):
    names = {"room": "config 2 'room' of BASELINE.json", "fig1": "config 3 'Figure-1-like' of BASELINE.json",
             "large": "config 5 'large' of BASELINE.json", "tiny": "config 1 'tiny' of BASELINE.json"}
    return {"workload": names[args.workload],
            "triangles": int(w.bvh.n_tris), "bvh_nodes": int(w.bvh.n_nodes), "K": int(w.K),
            "key_bits": int(w.key_bits), "diffuse_rays": int(n_d), "shadow_rays": int(n_s),
            "resolution": f"{w.width}x{w.height}x{w.spp}spp", "bounce": int(getattr(args, "bounce", 1)), "l2": l2,
            "parallelism": f"rays sharded over {args.gpus} GPU(s), BVH and cut replicated, no collective"}


# ------------------------------------------------------------------------------------------
def run_ours(args):
    import torch
    import torch.distributed as dist
    import hcc_inputs
    from paper_2305_16652_b200 import build as cuda_build
    cuda_build.build()
    import paper_2305_16652_b200 as hcc

    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if not torch.cuda.is_available():
        raise SystemExit("bench.py needs a CUDA device: the product path has no CPU fallback")
    torch.cuda.set_device(local)
    if world > 1:
        dist.init_process_group("nccl", device_id=torch.device("cuda", local))
    hbm_gbs, sm_max_mhz, peak_kind = _peaks()

    # ---- inputs (seeded; rank r draws its own sub-pixel samples of the same scene)
    w = hcc_inputs.Workload(args.workload, rank=rank, res_scale=args.res_scale)
    b = w.bvh
    bvh = hcc.Bvh(b.nodes, b.tris, b.prim_idx)

    def gpu_trace_closest(_bvh, rays):
        h = hcc.trace(bvh, torch.from_numpy(rays).cuda(), None, hcc.TRACE_CLOSEST)
        t, p, _, _ = hcc.hits_to_numpy(h)
        return t, p
    diffuse_h, shadow_h = w.first_bounce(gpu_trace_closest)
    for b_i in range(2, args.bounce + 1):      # later bounces: trace the previous diffuse batch, spawn the next
        t_prev, p_prev = gpu_trace_closest(None, diffuse_h)
        diffuse_h, shadow_h, _ = w.bounce(b_i, diffuse_h, t_prev, p_prev)
    n_d, n_s = diffuse_h.shape[0], shadow_h.shape[0]
    n = n_d + n_s
    diffuse = torch.from_numpy(diffuse_h).cuda()
    shadow = torch.from_numpy(shadow_h).cuda()
    batches = ((diffuse, hcc.TRACE_CLOSEST, "diffuse"), (shadow, hcc.TRACE_ANY, "shadow"))

    # ---- pre-process (once per scene): density + cut
    ev = lambda: torch.cuda.Event(enable_timing=True)
    had = hcc.density(bvh)
    cut = hcc.select_cut(bvh, had, w.K, w.key_bits)
    torch.cuda.synchronize()
    e0, e1 = ev(), ev()
    e0.record()
    hcc.density(bvh, out=had)
    hcc.select_cut(bvh, had, w.K, w.key_bits, cut=cut)
    e1.record()
    torch.cuda.synchronize()
    cut_ms = e0.elapsed_time(e1)
    info = cut.info()
    container = info["container_bits"]
    passes = (info["bits_used"] + 7) // 8

    pipe = hcc.Pipeline(max(n_d, n_s), 64, host_staging=True)
    hits_d = torch.empty((n_d, 4), dtype=torch.float32, device="cuda")
    hits_s = torch.empty(n_s, dtype=torch.uint8, device="cuda")
    hits = {"diffuse": hits_d, "shadow": hits_s}
    flush = torch.empty(256 * 1024 * 1024 // 4, dtype=torch.int32, device="cuda")   # 256 MiB > 126 MB L2

    def step(order):
        for rays, mode, name in batches:
            pipe.reorder_trace(bvh, cut, order, rays, mode, hits=hits[name], key_bits=w.key_bits)

    def timed(order, steps, warmup, per_stage=False):
        for _ in range(warmup):
            step(order)
        torch.cuda.synchronize()
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()
        pairs = [(ev(), ev()) for _ in range(steps)]
        stage = {nm: {"encode": 0.0, "sort": 0.0, "trace": 0.0} for _, _, nm in batches}
        t0 = time.time()
        for s, e in pairs:
            flush.zero_()                       # L2 flush, outside the event bracket
            s.record()
            if per_stage:
                for rays, mode, name in batches:
                    pipe.reorder_trace(bvh, cut, order, rays, mode, hits=hits[name], key_bits=w.key_bits)
                    ms = pipe.stage_ms()
                    for k in stage[name]:
                        stage[name][k] += ms[k] / steps
            else:
                step(order)
            e.record()
        torch.cuda.synchronize()
        t1 = time.time()
        if world > 1:
            dist.barrier()
        ms = sum(s.elapsed_time(e) for s, e in pairs)
        if world > 1:
            t = torch.tensor([ms], dtype=torch.float64, device="cuda")
            dist.all_reduce(t, op=dist.ReduceOp.MAX)
            ms = float(t.item())
        return ms / steps, stage, (t0, t1)

    # ---- the timed region: K steps of the HCC-ordered hot path
    sampler = ClockSampler(local)
    if rank == 0:
        sampler.start()
        time.sleep(0.3)
    ms_step, _, (t0, t1) = timed(hcc.ORDER_HCC, args.steps, args.warmup)
    clocks = sampler.stop(t0, t1) if rank == 0 else None
    value = world * n / (ms_step * 1e-3) / 1e6

    # ---- stage split and the comparison orders on the same rays (short runs, same hygiene)
    k_cmp = max(3, min(args.steps, 10))
    orders = {}
    for name, order in (("hcc", hcc.ORDER_HCC), ("twopoint", hcc.ORDER_TWOPOINT), ("nosort", hcc.ORDER_NOSORT)):
        ms, stage, _ = timed(order, k_cmp, 3, per_stage=True)
        o = {"ms_per_step": ms, "mrays_per_s_incl": n / ms / 1e3}
        for bn, nb in (("diffuse", n_d), ("shadow", n_s)):
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

    # ---- the same step with the two batches of the bounce on two streams (one pipeline each): the encode and
    #      the latency-bound sort of one batch fill issue slots the other batch's traversal leaves idle.
    #      Reported beside `value`, which stays the plain one-stream step.
    pipe2 = hcc.Pipeline(n_d, 64)
    streams_o = (torch.cuda.Stream(), torch.cuda.Stream())

    def step_overlapped():
        cur = torch.cuda.current_stream()
        for st in streams_o:
            st.wait_stream(cur)
        # shadow (the longer batch) first
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
    ov_ms = float(np.mean(ov))
    if world > 1:
        t = torch.tensor([ov_ms], dtype=torch.float64, device="cuda")
        dist.all_reduce(t, op=dist.ReduceOp.MAX)
        ov_ms = float(t.item())
    overlapped = {"ms_per_step": ov_ms, "value": world * n / ov_ms / 1e3, "unit": UNIT,
                  "how": "diffuse and shadow batch of the step on two streams, one hcc_pipeline each"}

    # ---- trace work counters (instrumented kernel, never timed) and ANC, HCC order
    diag = {}
    alu_peak = SM_COUNT * LANES_PER_SM * sm_max_mhz * 1e6 / 1e12     # T lane-op/s
    for rays, mode, name in batches:
        keys = hcc.encode(rays, cut)
        keys0 = keys.clone()
        perm = hcc.sort(keys, info["bits_used"])
        st = hcc.trace_stats(bvh, rays, perm, mode)
        st0 = hcc.trace_stats(bvh, rays, None, mode)
        ops = (st["nodes"] * OPS_NODE + st["tris"] * OPS_TRI)
        diag[name] = {"anc_hcc": hcc.anc(keys0, perm), "anc_nosort": hcc.anc(keys0, None),
                      "node_bytes_per_ray": st["node_bytes_per_ray"], "tri_bytes_per_ray": st["tri_bytes_per_ray"],
                      "node_bytes_per_ray_nosort": st0["node_bytes_per_ray"], "max_stack": st["max_stack"],
                      "lane_ops_per_ray": ops / rays.shape[0], "lane_ops": ops}
    nrays = {"diffuse": n_d, "shadow": n_s}
    key_b = container // 8
    stages = {}
    for name in ("diffuse", "shadow"):
        o, nb = orders["hcc"][name], nrays[name]
        enc_bytes = nb * (32 + key_b)
        sort_bytes = nb * (key_b + passes * 2 * (key_b + 4))
        enc_gbs = enc_bytes / (o["encode_ms"] * 1e-3) / 1e9
        sort_gbs = sort_bytes / (o["sort_ms"] * 1e-3) / 1e9
        tr = diag[name]["lane_ops"] / (o["trace_ms"] * 1e-3) / 1e12
        enc_ops = nb * info["bits_used"] * OPS_BOX / (o["encode_ms"] * 1e-3) / 1e12
        stages[name] = {
            "encode": {"bound": "hbm", "achieved": enc_gbs, "peak": hbm_gbs, "unit": "GB/s", "frac": enc_gbs / hbm_gbs,
                       "alu_achieved_tlaneops": enc_ops, "alu_frac": enc_ops / alu_peak, "box_tests_per_ray": info["bits_used"]},
            "sort": {"bound": "hbm", "achieved": sort_gbs, "peak": hbm_gbs, "unit": "GB/s", "frac": sort_gbs / hbm_gbs,
                     "passes": passes},
            "trace": {"bound": "alu", "achieved": tr, "peak": alu_peak, "unit": "Tlaneop/s", "frac": tr / alu_peak}}
    # dominant kernel of the step = the closest-hit traversal of the diffuse batch
    dom = max((("diffuse", "trace"), ("shadow", "trace"), ("diffuse", "sort"), ("shadow", "sort"),
               ("diffuse", "encode"), ("shadow", "encode")), key=lambda k: orders["hcc"][k[0]][k[1] + "_ms"])
    roof = dict(stages[dom[0]][dom[1]])
    roof = {"bound": roof["bound"], "achieved": roof["achieved"], "peak": roof["peak"], "unit": roof["unit"],
            "frac": roof["frac"],
            "traffic": NCU_TRAFFIC_ROOM[dom[0]] if (args.workload == "room" and dom[1] == "trace" and args.bounce == 1 and args.res_scale == 1.0) else None,
            "traffic_unit": "bytes per launch (dram read + write, ncu, profiles/r1b_ncu_full.md)",
            "kernel": f"{dom[1]} ({dom[0]} batch)",
            "peak_source": (f"{peak_kind} HBM copy" if roof["bound"] == "hbm" else
                            f"148 SMs x 128 fp32 lanes x {sm_max_mhz:.0f} MHz (DESIGN.md)")}

    # ---- encode and sort at the batch size of configs 3/5 (the shadow batch tiled to ~33.5 M rays): the
    #      config-2 batches (1-2 M pairs) are launch- and latency-bound, so the HBM fractions that the
    #      north_star's 60 % bar is about are measured here (SURVEY.md §7 "hard parts", §8(d))
    large = None
    if world == 1 and not args.no_large_n:
        reps = max(1, (1 << 25) // n_s)
        big = shadow.repeat(reps, 1) if reps > 1 else shadow
        nb = big.shape[0]
        keys_b = hcc.encode(big, cut)
        keys_b0 = keys_b.clone()
        ws_b = torch.empty(hcc.sort_workspace_bytes(nb, container), dtype=torch.uint8, device="cuda")
        perm_b = torch.empty(nb, dtype=torch.int32, device="cuda")

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
        enc_ms = med(lambda: hcc.encode(big, cut, keys=keys_b))
        sort_ms = med(lambda: hcc.sort(keys_b, info["bits_used"], perm=perm_b, workspace=ws_b), setup=lambda: keys_b.copy_(keys_b0))
        tp_keys = hcc.encode_twopoint(big, bvh.scene_lo, bvh.scene_hi, w.key_bits)
        tp_ms = med(lambda: hcc.encode_twopoint(big, bvh.scene_lo, bvh.scene_hi, w.key_bits, keys=tp_keys))
        tp_keys0 = tp_keys.clone()
        tp_bits_used = 6 * (w.key_bits // 6)
        tp_cb = 32 if w.key_bits <= 32 else 64
        tp_passes = (tp_bits_used + 7) // 8
        ws_t = torch.empty(hcc.sort_workspace_bytes(nb, tp_cb), dtype=torch.uint8, device="cuda")
        perm_t = torch.empty(nb, dtype=torch.int32, device="cuda")
        tp_sort_ms = med(lambda: hcc.sort(tp_keys, tp_bits_used, perm=perm_t, workspace=ws_t), setup=lambda: tp_keys.copy_(tp_keys0))
        tp_sort_bytes = nb * (tp_cb // 8 + tp_passes * 2 * (tp_cb // 8 + 4))
        kb = container // 8
        eb, sb_ = nb * (32 + kb), nb * (kb + passes * 2 * (kb + 4))
        tkb = 4 if w.key_bits <= 32 else 8
        large = {"rays": int(nb), "how": f"shadow batch tiled x{reps}",
                 "encode": {"ms": enc_ms, "bound": "hbm", "achieved": eb / enc_ms / 1e6, "peak": hbm_gbs, "unit": "GB/s",
                            "frac": eb / enc_ms / 1e6 / hbm_gbs,
                            "alu_frac": nb * info["bits_used"] * OPS_BOX / (enc_ms * 1e-3) / 1e12 / (SM_COUNT * LANES_PER_SM * sm_max_mhz * 1e6 / 1e12)},
                 "sort": {"ms": sort_ms, "bound": "hbm", "achieved": sb_ / sort_ms / 1e6, "peak": hbm_gbs, "unit": "GB/s",
                          "frac": sb_ / sort_ms / 1e6 / hbm_gbs, "passes": passes},
                 "sort_twopoint_keys": {"ms": tp_sort_ms, "bound": "hbm", "achieved": tp_sort_bytes / tp_sort_ms / 1e6, "peak": hbm_gbs,
                                        "unit": "GB/s", "frac": tp_sort_bytes / tp_sort_ms / 1e6 / hbm_gbs, "passes": tp_passes,
                                        "note": "well-spread Morton digits: the per-bit ballot path of the sort"},
                 "encode_twopoint": {"ms": tp_ms, "bound": "hbm", "achieved": nb * (32 + tkb) / tp_ms / 1e6, "peak": hbm_gbs,
                                     "unit": "GB/s", "frac": nb * (32 + tkb) / tp_ms / 1e6 / hbm_gbs}}
        del big, keys_b, keys_b0, ws_b, perm_b, tp_keys, tp_keys0, ws_t, perm_t
        torch.cuda.empty_cache()

    # ---- studies, on request: f1 sort truncation, f2 lambda and
    #      ANC, f3 prefix path code (:116-128), f4 regular grid (:243)
    studies = None
    if args.studies and world == 1:
        def med_ms(fn, setup=None, k=5):
            out = []
            for i in range(k + 1):
                if setup:
                    setup()
                flush.zero_()
                s0, e0 = ev(), ev()
                s0.record(); fn(); e0.record()
                torch.cuda.synchronize()
                if i >= 1:
                    out.append(s0.elapsed_time(e0))
            return float(np.median(out))

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
        # the same rays in a SHUFFLED input order (a wavefront renderer does not emit rays in camera order):
        # the regime in which reordering has something to gain
        saved = batches
        g = torch.Generator(device="cuda").manual_seed(0x5EED)
        batches = tuple((rays[torch.randperm(rays.shape[0], device="cuda", generator=g)].contiguous(), mode, name)
                        for rays, mode, name in saved)
        studies["orders_shuffled_input"] = {
            "nosort": run_order(None, 0),
            "twopoint": run_order(lambda rays, keys=None: hcc.encode_twopoint(rays, bvh.scene_lo, bvh.scene_hi, w.key_bits, keys=keys), tp_bits),
            "hcc": run_order(hcc_keys(cut), info["bits_used"])}
        batches = saved
        step(hcc.ORDER_HCC)          # the hit buffers hold the unshuffled batches' results again (checked by the e2e leg)
        studies["note"] = ("per batch medians of 5; grid = regular-grid tables of the same widths through the same encoder; "
                           "ppc = prefix path code with key_bits tests (upper-bound ordering, PAPER.md:128)")

    # ---- e2e: the same step through the C ABI with HOST buffers (pinned), copies inside the timing
    rays_pin = {"diffuse": torch.from_numpy(diffuse_h).pin_memory(), "shadow": torch.from_numpy(shadow_h).pin_memory()}
    hits_pin = {"diffuse": torch.empty((n_d, 4), dtype=torch.float32).pin_memory(),
                "shadow": torch.empty(n_s, dtype=torch.uint8).pin_memory()}

    # one pipeline and one stream per batch: the shadow batch's host->device copy overlaps the diffuse
    # batch's kernels, the diffuse hits go back while the shadow batch is traced
    pipes_h = {"diffuse": hcc.Pipeline(n_d, 64, host_staging=True), "shadow": pipe}
    streams_h = {"diffuse": torch.cuda.Stream(), "shadow": torch.cuda.Stream()}

    def step_host():
        cur = torch.cuda.current_stream()
        for _, mode, name in batches:
            st = streams_h[name]
            st.wait_stream(cur)
            pipes_h[name].reorder_trace_host_async(bvh, cut, hcc.ORDER_HCC, rays_pin[name], hits_pin[name], mode,
                                                   key_bits=w.key_bits, stream=st)
        for name in ("diffuse", "shadow"):
            pipes_h[name].synchronize()
            cur.wait_stream(streams_h[name])
    for _ in range(3):
        step_host()
    torch.cuda.synchronize()
    if world > 1:
        dist.barrier()
    k_e2e = max(3, min(args.steps, 10))
    e2e_ms = 0.0
    for _ in range(k_e2e):
        flush.zero_()
        s, e = ev(), ev()
        s.record()
        step_host()
        e.record()
        torch.cuda.synchronize()
        e2e_ms += s.elapsed_time(e) / k_e2e
    if world > 1:
        t = torch.tensor([e2e_ms], dtype=torch.float64, device="cuda")
        dist.all_reduce(t, op=dist.ReduceOp.MAX)
        e2e_ms = float(t.item())
    assert torch.equal(hits_pin["shadow"].cuda(), hits_s) and torch.equal(hits_pin["diffuse"].cuda().view(torch.int32), hits_d.view(torch.int32))
    e2e = {"value": world * n / e2e_ms / 1e3, "unit": UNIT, "ms_per_step": e2e_ms,
           "h2d_bytes_per_step": 32 * n, "d2h_bytes_per_step": 16 * n_d + n_s}

    # kernels launched per step: per batch 1 key kernel + (histogram + scan + one per digit) + 1 trace
    launches_per_step = 2 * (1 + (2 + passes) + 1)

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
            "config": _config(args, w, n_d, n_s, l2="flushed between timed steps (256 MiB write)"),
            "clocks": clocks, "e2e": e2e, "gpu_launches": launches_per_step * args.steps,
            "roofline": roof, "cpu_baseline": cpu,
            "cut": {"widths": info["widths"], "K_eff": info["K_eff"], "bits_used": info["bits_used"],
                    "container_bits": container, "cut_ms": cut_ms},
            "orders": orders, "speedup_hcc": speed, "stages_roofline_hcc": stages, "stages_roofline_large_batch": large, "two_stream_step": overlapped, "studies": studies,
            "diagnostics": diag,
            "paper_context": "RTX 3060, Breakfast: HCC 67.6 vs NoSort 37.4 vs TwoPoint 56.8 Mrays/s trace-only (PAPER.md:294-299); not comparable"}
    print(json.dumps(line))
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
    ap.add_argument("--studies", action="store_true", help="add the NEXT-row studies: sort truncation, lambda/ANC, grid and PPC orders")
    ap.add_argument("--no-large-n", action="store_true", help="skip the large-batch encode/sort roofline leg")
    args = ap.parse_args()
    if args.warmup < 3 and args.impl == "ours":
        args.warmup = 3
    return run_reference(args) if args.impl == "reference" else run_ours(args)


if __name__ == "__main__":
    sys.exit(main())
