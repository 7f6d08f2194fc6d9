"""N > 1 plumbing of bench.py on CPU: world_size-2 gloo.  The path has no exchange step (DESIGN.md section 8:
replicas only), so what is covered is rank-dependent input seeding, max-over-ranks timing and the aggregate."""
import os
import socket

import numpy as np
import pytest

torch = pytest.importorskip("torch")
import torch.distributed as dist
import torch.multiprocessing as mp


def _free_port():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def _worker(rank, world, port, out):
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(world))
    import bench
    dist.init_process_group("gloo", rank=rank, world_size=world)
    try:
        _, _, cells = bench.make_inputs(256, rank)
        fake_ms = 10.0 * (rank + 1)               # rank 1 is the slow one
        ms = bench.max_over_ranks(dist, fake_ms)
        val = bench.aggregate_value(world, 256, ms)
        sums = torch.tensor([float(cells.T.sum())], dtype=torch.float64)
        gathered = [torch.zeros_like(sums) for _ in range(world)]
        dist.all_gather(gathered, sums)
        dist.barrier()
        if rank == 0:
            out.put((ms, val, [float(g.item()) for g in gathered]))
    finally:
        dist.destroy_process_group()


def test_two_rank_replicas_gloo():
    world, port = 2, _free_port()
    ctx = mp.get_context("spawn")
    out = ctx.Queue()
    procs = [ctx.Process(target=_worker, args=(r, world, port, out)) for r in range(world)]
    for p in procs:
        p.start()
    ms, val, sums = out.get(timeout=180)
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    assert ms == 20.0                              # max over ranks, not rank 0's own 10 ms
    assert val == pytest.approx(2 * 256 / 20e-3)   # whole-job aggregate, weak scaling
    assert sums[0] != sums[1]                      # each replica draws its own cells


def test_single_rank_helpers():
    import bench
    assert bench.max_over_ranks(None, 3.5) == 3.5
    assert bench.aggregate_value(1, 1000, 2.0) == pytest.approx(5e5)
    pk = bench.peaks()
    assert pk["bf16"] > 0 and pk["hbm"] > 0
