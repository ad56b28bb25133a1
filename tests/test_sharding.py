"""Multi-process (gloo, world_size 2, CPU) test of the N > 1 host logic of bench.py / DESIGN.md
section 8: the path shards with no data-path collective -- every rank owns a contiguous range of
supernovae balanced by observation count, the only exchanges are the barrier and the max-over-ranks
of the timing.  The per-rank 'compute' here is a pure index/bookkeeping stand-in (the CUDA path
cannot run on a CPU box and the oracle is not part of the product path)."""
import os
import socket

import numpy as np
import torch
import torch.distributed as dist
import torch.multiprocessing as mp

import workloads


def _free_port():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def _worker(rank, world, port, q):
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(world))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    try:
        wl = workloads.make_workload(2, n_sn=101, ragged=True)
        n_obs = np.diff(wl.obs_offset)
        bounds = workloads.shard_bounds(wl.n_sn, n_obs, world)
        lo, hi = bounds[rank], bounds[rank + 1]
        shard = workloads.subset(wl, np.arange(lo, hi))
        # shard-local work: one value per owned supernova (stand-in for chi^2), no communication
        local = np.array([float(np.sum(shard.time[shard.obs_offset[i]:shard.obs_offset[i + 1]])) for i in range(shard.n_sn)])
        # timing protocol of bench.py: barrier, per-rank time, MAX over ranks
        dist.barrier()
        t = torch.tensor([1.0 + rank], dtype=torch.float64)
        dist.all_reduce(t, op=dist.ReduceOp.MAX)
        # optional single exchange step: gather the per-unit vectors on rank 0
        sizes = [torch.zeros(1, dtype=torch.int64) for _ in range(world)]
        dist.all_gather(sizes, torch.tensor([shard.n_sn], dtype=torch.int64))
        pad = int(max(s.item() for s in sizes))
        buf = torch.zeros(pad, dtype=torch.float64)
        buf[:shard.n_sn] = torch.from_numpy(local)
        parts = [torch.zeros(pad, dtype=torch.float64) for _ in range(world)]
        dist.all_gather(parts, buf)
        if rank == 0:
            full = np.concatenate([p.numpy()[:int(s.item())] for p, s in zip(parts, sizes)])
            q.put((bounds, float(t.item()), full, int(shard.n_obs_total)))
        else:
            q.put((bounds, float(t.item()), None, int(shard.n_obs_total)))
    finally:
        dist.destroy_process_group()


def test_world2_contiguous_balanced_shards_and_max_time():
    world, port = 2, _free_port()
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    procs = [ctx.Process(target=_worker, args=(r, world, port, q)) for r in range(world)]
    for p in procs:
        p.start()
    res = [q.get(timeout=120) for _ in range(world)]
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    wl = workloads.make_workload(2, n_sn=101, ragged=True)
    bounds = res[0][0]
    assert bounds[0] == 0 and bounds[-1] == wl.n_sn and all(a <= b for a, b in zip(bounds, bounds[1:]))
    assert all(r[1] == 2.0 for r in res)  # max over ranks of (1 + rank)
    n_obs = np.diff(wl.obs_offset)
    per_rank = sorted(r[3] for r in res)
    assert sum(per_rank) == wl.n_obs_total
    assert abs(per_rank[0] - per_rank[1]) <= 2 * int(n_obs.max())  # balanced by observation count
    full = next(r[2] for r in res if r[2] is not None)
    want = np.array([float(np.sum(wl.time[wl.obs_offset[i]:wl.obs_offset[i + 1]])) for i in range(wl.n_sn)])
    assert np.array_equal(full, want)  # shards tile the supernovae exactly once, in order


def test_shard_bounds_edge_cases():
    assert workloads.shard_bounds(0, np.zeros(0), 4) == [0, 0, 0, 0, 0]
    assert workloads.shard_bounds(3, np.ones(3), 1) == [0, 3]
    b = workloads.shard_bounds(10, np.array([100] + [1] * 9), 2)
    assert b[0] == 0 and b[-1] == 10 and b[1] >= 1
    sub = workloads.subset(workloads.make_workload(2, n_sn=5), [3, 1])
    assert sub.n_sn == 2 and sub.n_obs_total == 120
