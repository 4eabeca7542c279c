"""Multi-GPU layout of the path: rays are independent in encode and trace and
the sort only has to create coherence within one GPU, so a batch is cut into contiguous ray
ranges (primary-sample order), one per rank; the BVH and the cut are replicated; there is no
collective on the data path.  Only a consumer that wants all hits in one place gathers them.

Host logic only (no arithmetic of the method); works with any torch.distributed backend.
"""
import torch
import torch.distributed as dist


def ray_shard(n, rank, world):
    """[start, stop) of rank's contiguous share of n rays; sizes differ by at most one and the
    shares tile [0, n) in rank order."""
    n, rank, world = int(n), int(rank), int(world)
    if world < 1 or not 0 <= rank < world or n < 0:
        raise ValueError("bad shard request")
    q, r = divmod(n, world)
    start = rank * q + min(rank, r)
    return start, start + q + (1 if rank < r else 0)


def gather_hits(local, n, group=None):
    """Reassemble per-rank result slices (first dimension = this rank's rays, in order) into the
    full [n, ...] tensor on every rank.  Slices may differ in length by one."""
    world = dist.get_world_size(group)
    rank = dist.get_rank(group)
    sizes = [ray_shard(n, r, world)[1] - ray_shard(n, r, world)[0] for r in range(world)]
    if local.shape[0] != sizes[rank]:
        raise ValueError("local slice does not match this rank's shard")
    m = max(sizes) if sizes else 0
    pad = torch.zeros((m,) + tuple(local.shape[1:]), dtype=local.dtype, device=local.device)
    pad[: local.shape[0]] = local
    parts = [torch.empty_like(pad) for _ in range(world)]
    dist.all_gather(parts, pad, group=group)
    return torch.cat([p[:s] for p, s in zip(parts, sizes)], 0)


def sharded_reorder_trace(pipe, bvh, cut, order, rays, mode, rank, world, key_bits=32, hits=None, stream=None):
    """This rank's share of one batch through the one-call hot path (hcc_reorder_trace): `rays` is the
    WHOLE batch on this rank's device ([n, 8] float32, replicated like the BVH and the cut); the rank
    encodes, sorts and traces rays[start:stop] only.  Returns (local hits, (start, stop)); the hits of
    ray start + i are at local index i.  No collective: gather_hits is for a consumer that wants them
    all in one place."""
    start, stop = ray_shard(rays.shape[0], rank, world)
    local = rays[start:stop]          # contiguous rows of 32 bytes: the slice keeps the 32-byte alignment
    out = pipe.reorder_trace(bvh, cut, order, local, mode, hits=hits, key_bits=key_bits, stream=stream)
    return out, (start, stop)
