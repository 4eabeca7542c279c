"""Multi-GPU host logic on CPU (gloo, world_size 2): contiguous ray shards tile the batch, and
per-shard results gathered in rank order equal the single-process result (rays are independent in
encode and trace).  The per-shard compute here is the oracle (tests may use it)."""
import os
import socket

import numpy as np
import pytest


def test_ray_shard_tiles_the_batch():
    from paper_2305_16652_b200.shard import ray_shard
    for n in (0, 1, 2, 7, 4096, 1048576 + 3):
        for world in (1, 2, 3, 8):
            spans = [ray_shard(n, r, world) for r in range(world)]
            assert spans[0][0] == 0 and spans[-1][1] == n
            assert all(a[1] == b[0] for a, b in zip(spans, spans[1:]))
            sizes = [b - a for a, b in spans]
            assert max(sizes) - min(sizes) <= 1
    with pytest.raises(ValueError):
        ray_shard(10, 2, 2)


def _free_port():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def _worker(rank, world, port, rays, nodes, prim_idx, tris, out):
    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    import torch
    import torch.distributed as dist
    import oracle
    from paper_2305_16652_b200.shard import gather_hits, ray_shard
    dist.init_process_group("gloo", rank=rank, world_size=world)
    try:
        a, b = ray_shard(rays.shape[0], rank, world)
        mine = rays[a:b]
        tables, _, _ = oracle.select_cut(nodes, 64, 32)
        keys = oracle.encode_hcc(mine, nodes, tables)
        perm = oracle.sort(keys)                       # coherence is created per shard
        t, p, _, _ = oracle.closest_bvh(np.ascontiguousarray(mine[perm]), nodes, prim_idx, tris)
        local = np.empty((b - a, 2), dtype=np.float64)
        local[perm, 0] = t                             # results land at the ray's own index
        local[perm, 1] = p
        full = gather_hits(torch.from_numpy(local), rays.shape[0])
        keys_full = gather_hits(torch.from_numpy(keys.astype(np.int64)), rays.shape[0])
        if rank == 0:
            out.put((full.numpy(), keys_full.numpy()))
    finally:
        dist.destroy_process_group()


def test_sharded_path_equals_single_process(tiny):
    import torch.multiprocessing as mp
    import oracle
    rays = tiny.diffuse[:1001]                         # odd size: shards of 501 and 500
    b = tiny.bvh
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    port = _free_port()
    procs = [ctx.Process(target=_worker, args=(r, 2, port, rays, b.nodes, b.prim_idx, b.tris, q)) for r in range(2)]
    for p in procs:
        p.start()
    full, keys_full = q.get(timeout=120)
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    t, prim, _, _ = oracle.closest_bvh(rays, b.nodes, b.prim_idx, b.tris)
    tables, _, _ = oracle.select_cut(b.nodes, 64, 32)
    assert np.array_equal(full[:, 0], t.astype(np.float64))
    assert np.array_equal(full[:, 1], prim.astype(np.float64))
    assert np.array_equal(keys_full.astype(np.uint64), oracle.encode_hcc(rays, b.nodes, tables))


@pytest.mark.gpu
@pytest.mark.parametrize("world", [1, 3])
def test_sharded_product_path_on_one_gpu(world, tiny):
    """The code path bench.py --gpus N runs per rank (shard.sharded_reorder_trace -> hcc_reorder_trace on the
    rank's contiguous range), on the single GPU of the test box: the shards of every rank of a `world`-rank job,
    run one after the other, tile the batch and reproduce the unsharded hits bit for bit; with a one-rank
    process group gather_hits returns the same tensor."""
    import torch
    import torch.distributed as dist
    import paper_2305_16652_b200 as hcc
    from paper_2305_16652_b200.shard import gather_hits, sharded_reorder_trace
    b = tiny.bvh
    bvh = hcc.Bvh(b.nodes, b.tris, b.prim_idx)
    cut = hcc.select_cut(bvh, hcc.density(bvh), 64, 32)
    for rays_h, mode in ((tiny.diffuse[:4001], hcc.TRACE_CLOSEST), (tiny.shadow[:8003], hcc.TRACE_ANY)):
        rays = torch.from_numpy(rays_h).cuda()
        n = rays.shape[0]
        pipe = hcc.Pipeline(n, 64)
        whole = hcc.trace(bvh, rays, None, mode)
        parts, spans = [], []
        for rank in range(world):
            local, span = sharded_reorder_trace(pipe, bvh, cut, hcc.ORDER_HCC, rays, mode, rank, world)
            parts.append(local.clone())
            spans.append(span)
        assert spans[0][0] == 0 and spans[-1][1] == n and all(a[1] == c[0] for a, c in zip(spans, spans[1:]))
        assert torch.equal(torch.cat(parts, 0).view(torch.uint8), whole.view(torch.uint8))
    if world == 1:
        os.environ["MASTER_ADDR"] = "127.0.0.1"
        os.environ["MASTER_PORT"] = str(_free_port())
        dist.init_process_group("nccl", rank=0, world_size=1, device_id=torch.device("cuda", 0))
        try:
            assert torch.equal(gather_hits(parts[0], n).view(torch.uint8), whole.view(torch.uint8))
        finally:
            dist.destroy_process_group()


@pytest.mark.gpu
def test_bench_two_ranks_code_path_on_one_gpu():
    """`python bench.py --gpus 2` starts its own two ranks (torch.distributed.run); with HCC_BENCH_SHARED_GPU=1 they share the
    test box's one GPU and talk over gloo (a code-path check, not a measurement: no rank's kernels wait on another's).  The line
    must come from two ranks, and the strong-scaling leg's gathered hits (product kernels on each rank's shard.ray_shard range)
    must equal the unsharded trace."""
    import json
    import subprocess
    import sys
    root = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
    env = dict(os.environ, HCC_BENCH_SHARED_GPU="1")
    for k in ("RANK", "WORLD_SIZE", "LOCAL_RANK", "MASTER_ADDR", "MASTER_PORT"):
        env.pop(k, None)
    r = subprocess.run([sys.executable, os.path.join(root, "bench.py"), "--gpus", "2", "--workload", "tiny", "--steps", "3", "--configs=",
                        "--no-studies", "--no-cpu-baseline", "--no-large-n", "--quick"], capture_output=True, text=True, env=env,
                       timeout=600, cwd=root)
    assert r.returncode == 0, r.stderr[-2000:]
    last = r.stdout.splitlines()[-1]
    assert last.startswith("{") and len(last) < 4096       # the driver parses the last line and keeps only stdout's tail
    line = json.loads(last)
    assert line["value"] > 0 and line["roofline"]["frac"] > 0 and line["e2e"]["value"] > 0
    assert line["n_gpus"] == 2 and line["config"]["shared_gpu_code_path_check"] is True
    s = line["strong_scaling"]
    assert s["ranks"] == 2 and s["scaling"] == "strong" and s["gathered_hits_equal_unsharded"] is True
    assert s["rays_total"] == line["config"]["diffuse_rays"] + line["config"]["shadow_rays"]
