"""N > 1 path on CPU: world_size-2 gloo run of the problem sharding (the only multi-GPU logic the
path has: independent problems, no data-path collective).  The per-rank build is the CPU oracle
on the tiny config, standing in for the CUDA batched build that a GPU box would call."""
import os

import numpy as np
import pytest
import torch
import torch.distributed as dist
import torch.multiprocessing as mp

from paper_2104_10000_b200 import inputs, sharding


def test_shard_problems_partition():
    for nb in (1, 2, 5, 512):
        for world in (1, 2, 3, 8):
            seen = sorted(b for r in range(world) for b in sharding.shard_problems(nb, world, r))
            assert seen == list(range(nb))
    with pytest.raises(ValueError):
        sharding.shard_problems(4, 2, 2)


def _worker(rank, world, port, nb, out):
    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    from oracle import landau_oracle as oracle
    wl = inputs.config(0)
    wl.components = [[inputs.Component(0, 1.0, 1.0 + 0.1 * b), inputs.Component(1, 1.0, 1.0, 0.05 * b)] for b in range(nb)]
    sp = oracle.build_space(wl.mesh, wl.order)
    f_all = torch.from_numpy(np.stack([inputs.nodal_f(wl, sp.dof_r, sp.dof_z, b) for b in range(nb)]))

    def build_fn(f_local):
        vals, Cf = [], []
        for f in f_local.numpy():
            _, v, c, _ = oracle.build_all(wl.mesh, wl.order, wl.species, f, 1.0, precision="d")
            vals.append(v); Cf.append(c)
        return torch.from_numpy(np.stack(vals)), torch.from_numpy(np.stack(Cf))

    mine, vals, Cf = sharding.build_sharded(build_fn, f_all)
    assert mine == list(range(rank, nb, world))
    allv, allc = sharding.gather_results(mine, vals, Cf, nb)
    # timing reduction used by bench.py: max over ranks
    t = torch.tensor([float(rank + 1)])
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    assert float(t) == float(world)
    if rank == 0:
        ref_v, ref_c = build_fn(f_all)
        out["ok"] = bool(torch.equal(allv, ref_v) and torch.equal(allc, ref_c))
    dist.barrier()
    dist.destroy_process_group()


def test_world_size_2_gloo_sharded_build_matches_serial():
    from oracle import landau_oracle
    landau_oracle.build()
    mgr = mp.Manager()
    out = mgr.dict()
    port = 29500 + (os.getpid() % 2000)
    mp.spawn(_worker, args=(2, port, 5, out), nprocs=2, join=True)
    assert out.get("ok") is True
