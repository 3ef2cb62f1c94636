"""N > 1 path on CPU (world_size 2, gloo): zones shard across ranks with no data-path collective
(DESIGN.md section 7); only results/timings are gathered.  The per-rank compute here is the
oracle standing in for burn_zones (tests may call it); what is tested is the host logic that
bench.py and a multi-GPU caller use: shard_range / shard_workload, gather, max-over-ranks."""
import os
import socket

import numpy as np
import torch
import torch.distributed as dist
import torch.multiprocessing as mp

import oracle
from paper_1711_06203_b200.sharding import shard_range, shard_workload
from workloads import make_workload


def _free_port():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def _worker(rank, world, port, out_path):
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(world))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    w = make_workload(1, zones=np.arange(0, 4096, 16))          # 256 zones
    rho, T, X, (lo, hi) = shard_workload(w.rho, w.T, w.X, rank, world)
    To, Xo, ns, cnt = oracle.burn(w.net, rho, T, np.ascontiguousarray(X), w.dt, w.rtol, w.atol, nthreads=1)
    # gather variable-size shards: pad to the largest shard
    nmax = max(shard_range(w.nz, r, world)[1] - shard_range(w.nz, r, world)[0] for r in range(world))
    buf = torch.zeros((w.net.nspec + 2, nmax), dtype=torch.float64)
    buf[0, : hi - lo] = torch.from_numpy(To)
    buf[1, : hi - lo] = torch.from_numpy(ns.astype(np.float64))
    buf[2:, : hi - lo] = torch.from_numpy(Xo)
    parts = [torch.zeros_like(buf) for _ in range(world)]
    dist.all_gather(parts, buf)
    tms = torch.tensor([10.0 + rank], dtype=torch.float64)       # max-over-ranks timing reduction
    dist.all_reduce(tms, op=dist.ReduceOp.MAX)
    steps = torch.tensor([float(cnt["nst"])], dtype=torch.float64)
    dist.all_reduce(steps, op=dist.ReduceOp.SUM)
    if rank == 0:
        cat = torch.cat([parts[r][:, : shard_range(w.nz, r, world)[1] - shard_range(w.nz, r, world)[0]]
                         for r in range(world)], dim=1).numpy()
        np.save(out_path, np.vstack([cat, np.full((1, cat.shape[1]), tms.item()),
                                     np.full((1, cat.shape[1]), steps.item())]))
    dist.barrier()
    dist.destroy_process_group()


def test_two_rank_shard_equals_single(tmp_path):
    out = str(tmp_path / "gathered.npy")
    mp.spawn(_worker, args=(2, _free_port(), out), nprocs=2, join=True)
    got = np.load(out)
    w = make_workload(1, zones=np.arange(0, 4096, 16))
    To, Xo, ns, cnt = oracle.burn(w.net, w.rho, w.T, w.X, w.dt, w.rtol, w.atol)
    assert np.array_equal(got[0], To)
    assert np.array_equal(got[1], ns.astype(np.float64))
    assert np.array_equal(got[2:4], Xo)
    assert got[4, 0] == 11.0                      # max over ranks
    assert got[5, 0] == float(cnt["nst"])         # counters sum over ranks
