"""N>1 path on CPU: environments are the independent units; every rank owns a
contiguous env range and there is no collective on the data path.  world_size-2 `gloo` run:
each rank evaluates its shard with the oracle (the GPU library cannot run here), the shards
are gathered ONLY for checking, and must reproduce the single-process result bit for bit; the
timing reduction bench.py uses (MAX over ranks) is exercised too."""
import os
import socket

import numpy as np
import torch
import torch.distributed as dist
import torch.multiprocessing as mp

from oracle import etac_oracle as O
from paper_2604_20295_b200 import workloads as W


def test_shard_envs_partition():
    for n, ws in [(4096, 8), (10, 3), (7, 8), (1, 2)]:
        spans = [W.shard_envs(n, ws, r) for r in range(ws)]
        assert spans[0][0] == 0 and spans[-1][1] == n
        assert all(a[1] == b[0] for a, b in zip(spans, spans[1:]))
        sizes = [hi - lo for lo, hi in spans]
        assert max(sizes) - min(sizes) <= 1


def _free_port():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def _worker(rank, world, port, n_envs, q):
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    wl = W.config2(seed=11, n_envs=n_envs)
    lo, hi = W.shard_envs(n_envs, world, rank)
    r = O.step(O.model_from_workload(wl), indenters=wl.indenters, envs=range(lo, hi))
    mine = torch.from_numpy(r["U"].reshape(hi - lo, -1))
    # checking only: gather variable-sized shards (pad to the largest)
    cap = max(b - a for a, b in (W.shard_envs(n_envs, world, k) for k in range(world)))
    pad = torch.zeros((cap, mine.shape[1]), dtype=mine.dtype)
    pad[: hi - lo] = mine
    got = [torch.zeros_like(pad) for _ in range(world)]
    dist.all_gather(got, pad)
    t = torch.tensor([1.0 + rank], dtype=torch.float64)       # "elapsed time" of this rank
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    if rank == 0:
        full = torch.cat([g[: b - a] for g, (a, b) in zip(got, (W.shard_envs(n_envs, world, k) for k in range(world)))])
        q.put((full.numpy(), float(t)))
    dist.barrier()
    dist.destroy_process_group()


def test_two_rank_env_sharding_reproduces_single_process():
    n_envs, world = 5, 2
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    port = _free_port()
    procs = [ctx.Process(target=_worker, args=(r, world, port, n_envs, q)) for r in range(world)]
    for p in procs:
        p.start()
    full, tmax = q.get(timeout=120)
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    wl = W.config2(seed=11, n_envs=n_envs)
    ref = O.step(O.model_from_workload(wl), indenters=wl.indenters)["U"].reshape(n_envs, -1)
    assert np.array_equal(full, ref)
    assert tmax == 2.0
