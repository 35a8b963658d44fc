"""Multi-rank host logic on CPU (gloo, world_size 2): the point partition covers the field exactly
once, shards of a flame-profile state concatenate to the same profile, and the max-over-ranks
timing reduction bench.py uses works.  The oracle stands in for the kernels here (the path is
pointwise, so evaluating shards separately must equal evaluating the whole field)."""
import os
import socket

import numpy as np
import pytest
import torch
import torch.distributed as dist
import torch.multiprocessing as mp

from paper_2409_06404_b200 import shard
from paper_2409_06404_b200 import workloads as wl


def test_element_partition_is_exact():
    for ne in (0, 1, 7, 4096, 32768, 1000):
        for world in (1, 2, 3, 8):
            spans = [shard.element_range(ne, r, world) for r in range(world)]
            assert spans[0][0] == 0 and spans[-1][1] == ne
            assert all(a[1] == b[0] for a, b in zip(spans, spans[1:]))
            sizes = [b - a for a, b in spans]
            assert max(sizes) - min(sizes) <= 1
            assert shard.point_range(ne, world - 1, world)[1] == ne * 512
    with pytest.raises(ValueError):
        shard.element_range(8, 2, 2)
    assert shard.weak_range(1024, 1, 2) == (1024, 1024, 2048)


def _free_port():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def _worker(rank, world, port, q):
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    from oracle import crf_oracle
    n_elem = 6
    a, b = shard.point_range(n_elem, rank, world)
    total = n_elem * 512
    st = wl.make_state("C4", n=b - a, offset=a, total=total)
    o = crf_oracle.Oracle(wl.make_mechanism("C4"))
    r = o.production_rates(**st)
    # every rank's partial mass-conservation residual and point count, reduced without any data exchange
    W = torch.tensor(wl.make_mechanism("C4")["W"])
    resid = torch.tensor([float(np.max(np.abs(W.numpy() @ r["omega"]) / (W.numpy() @ r["S_omega"]))), float(b - a)])
    t = torch.tensor([0.010 * (rank + 1)], dtype=torch.float64)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    gathered = [torch.zeros(2, dtype=torch.float64) for _ in range(world)]
    dist.all_gather(gathered, resid.double())
    # profile continuity: the noise-free part of T of this shard equals that slice of the whole field
    x = (a + np.arange(b - a) + 0.5) / total
    q.put((rank, float(t.item()), [g.tolist() for g in gathered], float(st["T"].mean()), x[0], x[-1]))
    dist.barrier()
    dist.destroy_process_group()


def test_two_rank_sharding_gloo(oracle_mod):
    world, port = 2, _free_port()
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    procs = [ctx.Process(target=_worker, args=(r, world, port, q)) for r in range(world)]
    for p in procs:
        p.start()
    res = sorted(q.get(timeout=180) for _ in range(world))
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    for rank, tmax, gathered, _, _, _ in res:
        assert tmax == pytest.approx(0.020)               # max over ranks
        assert sum(g[1] for g in gathered) == 6 * 512     # shards cover the field exactly once
        assert all(g[0] <= 1e-12 for g in gathered)       # each shard conserves mass on its own
    assert res[0][5] < res[1][4]                          # rank 0's profile positions precede rank 1's
    assert res[0][3] < res[1][3]                          # flame profile: rank 1 holds the burnt side
