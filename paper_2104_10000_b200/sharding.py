"""Multi-GPU sharding of the batched build: independent problems, round-robin over ranks.

The path shards only over the batch dimension ("each configuration space point
advances the collision operator independently"); there is NO data-path collective.  One process
per GPU; `torch.distributed` is used for the optional gather of results and for timing barriers.
"""
from __future__ import annotations


def shard_problems(nproblems: int, world_size: int, rank: int) -> list[int]:
    """Problem indices owned by `rank`: b with b % world_size == rank (every problem exactly once)."""
    if not (0 <= rank < world_size):
        raise ValueError("rank out of range")
    return list(range(rank, nproblems, world_size))


def build_sharded(build_fn, f_all, group=None):
    """Runs build_fn(f_local) -> (vals_local, Cf_local) on this rank's problems of f_all[nb][S][n]
    and returns the local results with their problem indices.  build_fn is the batched build
    (LandauContext.jacobian_batched on a GPU box)."""
    import torch.distributed as dist
    world = dist.get_world_size(group) if dist.is_initialized() else 1
    rank = dist.get_rank(group) if dist.is_initialized() else 0
    mine = shard_problems(f_all.shape[0], world, rank)
    vals, Cf = build_fn(f_all[mine])
    return mine, vals, Cf


def gather_results(mine, vals, Cf, nproblems: int, group=None):
    """All-gathers the per-rank results into problem order (for checks; a solver would keep each
    problem's matrix on the rank that owns it).  Tensors must live where the backend can reach
    them (CPU for gloo, CUDA for nccl)."""
    import torch
    import torch.distributed as dist
    world = dist.get_world_size(group)
    out_v = torch.zeros((nproblems,) + tuple(vals.shape[1:]), dtype=vals.dtype, device=vals.device)
    out_c = torch.zeros((nproblems,) + tuple(Cf.shape[1:]), dtype=Cf.dtype, device=Cf.device)
    per = (nproblems + world - 1) // world
    pad_v = torch.zeros((per,) + tuple(vals.shape[1:]), dtype=vals.dtype, device=vals.device)
    pad_c = torch.zeros((per,) + tuple(Cf.shape[1:]), dtype=Cf.dtype, device=Cf.device)
    pad_v[: len(mine)] = vals
    pad_c[: len(mine)] = Cf
    all_v = [torch.zeros_like(pad_v) for _ in range(world)]
    all_c = [torch.zeros_like(pad_c) for _ in range(world)]
    dist.all_gather(all_v, pad_v, group=group)
    dist.all_gather(all_c, pad_c, group=group)
    for r in range(world):
        idx = shard_problems(nproblems, world, r)
        out_v[idx] = all_v[r][: len(idx)]
        out_c[idx] = all_c[r][: len(idx)]
    return out_v, out_c
