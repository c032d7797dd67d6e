"""world_size-2 gloo tests (CPU) of the multi-GPU host logic: batch-member sharding with no data-path collective and
the max-over-ranks timing reduction of bench.py.  Each rank evaluates its own members with the
oracle; gathering the shards must reproduce the unsharded batch exactly (members are independent)."""
import os
import socket

import numpy as np
import pytest
import torch
import torch.distributed as dist
import torch.multiprocessing as mp

import fe_inputs as fi
from oracle import fe_oracle as orc
from gpu_util import oracle_problem
from paper_2605_28800_b200.parallel import owner_of, reduce_timing, shard_members, throughput


def test_shard_members_partition():
    for batch in (0, 1, 4, 5, 16, 17):
        for world in (1, 2, 3, 8):
            seen = []
            for r in range(world):
                s = shard_members(batch, r, world)
                seen += list(s)
                assert abs(len(s) - batch / world) < 1
            assert seen == list(range(batch))
            for m in range(batch):
                assert m in shard_members(batch, owner_of(m, batch, world), world)
    with pytest.raises(ValueError):
        shard_members(4, 2, 2)


def test_reduce_timing_single_process():
    assert reduce_timing(3.0, 7.0) == (3.0, 7.0)
    v, ms = throughput(2.0, 10.0)
    assert ms == 2.0 and v == 10.0 / 2e-3


def _free_port():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def _worker(rank, world, port, out):
    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    try:
        w = fi.config3(n=8, batch=5)                      # 5 members at different temperatures
        mine = shard_members(w.batch, rank, world)
        rhs = np.zeros((w.batch, 3, 8, 8, 8))
        for b in mine:
            rhs[b] = orc.Oracle(oracle_problem(w, b), elec="fft").rhs(w.P0[b])
        t = torch.from_numpy(rhs)
        dist.all_reduce(t, op=dist.ReduceOp.SUM)          # test-side gather only: shards are disjoint
        ms, units = reduce_timing(10.0 * (rank + 1), float(len(mine) * w.cells))
        val, ms2 = throughput(10.0 * (rank + 1), float(len(mine) * w.cells))
        if rank == 0:
            out.put((t.numpy(), ms, units, val, ms2, list(mine)))
        dist.barrier()
    finally:
        dist.destroy_process_group()


def test_two_ranks_gloo_shards_reproduce_the_batch():
    world = 2
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    port = _free_port()
    procs = [ctx.Process(target=_worker, args=(r, world, port, q)) for r in range(world)]
    for p in procs:
        p.start()
    got, ms, units, val, ms2, mine0 = q.get(timeout=120)
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    w = fi.config3(n=8, batch=5)
    assert mine0 == [0, 1, 2]
    for b in range(w.batch):
        want = orc.Oracle(oracle_problem(w, b), elec="fft").rhs(w.P0[b])
        assert np.array_equal(got[b], want)               # same code, same inputs: bit-identical
    assert ms == 20.0 and ms2 == 20.0                     # slowest rank
    assert units == 5 * w.cells
    assert val == units / 20e-3
