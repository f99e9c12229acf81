"""N > 1 host logic on CPU: world_size-2 gloo run of paper_1910_08448_b200.sharding.

The path shards by independent problems: no data-path collective, only the
measurement is reduced (max of the durations, sum of the units and launches).  These tests start
two real processes over gloo on 127.0.0.1 and check exactly that, plus the seed assignment.
No GPU, no kernel call.
"""
import os
import socket

import pytest
import torch
import torch.distributed as dist
import torch.multiprocessing as mp

from paper_1910_08448_b200 import inputs, sharding


def _free_port():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def _worker(rank, world, port, out):
    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    try:
        c = inputs.CONFIGS[1]
        rp = sharding.rank_problem(c.field_seed, c.mpr_seed, rank, world)
        values, mask, _ = inputs.make_problem(c.L, c.xi, rp.field_seed, c.f, c.lognormal)
        n_free = int(mask.sum())
        # a rank-dependent duration and launch count: rank 1 is the slow one
        ms, launches, sweeps = 10.0 + 5.0 * rank, 100 + rank, 200
        units = 2.0 * n_free * sweeps
        ms_max, units_total, launches_total = sharding.aggregate(ms, units, launches, world)
        # each rank also publishes what it contributed, so the parent can re-add it
        mine = torch.tensor([float(rp.field_seed), float(rp.mpr_seed), units, float(values[mask == 0].sum())],
                            dtype=torch.float64)
        gathered = [torch.zeros_like(mine) for _ in range(world)]
        dist.all_gather(gathered, mine)
        out[rank] = (ms_max, units_total, launches_total, [g.tolist() for g in gathered])
    finally:
        dist.destroy_process_group()


@pytest.mark.timeout(180)
def test_two_ranks_reduce_max_time_and_sum_units():
    world, port = 2, _free_port()
    with mp.Manager() as mgr:
        out = mgr.dict()
        mp.spawn(_worker, args=(world, port, out), nprocs=world, join=True)
        res = dict(out)
    assert set(res) == {0, 1}
    # every rank holds the same reduced triple
    assert res[0][:3] == res[1][:3]
    ms_max, units_total, launches_total, gathered = res[0]
    assert ms_max == 15.0                                  # the slow rank decides
    assert launches_total == 100 + 101
    assert units_total == gathered[0][2] + gathered[1][2]  # sum of what each rank did
    # distinct problems per rank: seeds differ, and so do the generated fields
    c = inputs.CONFIGS[1]
    assert gathered[0][0] == c.field_seed and gathered[0][1] == c.mpr_seed   # rank 0 = BASELINE's seeds
    assert gathered[1][0] == c.field_seed + sharding.FIELD_SEED_STRIDE
    assert gathered[1][1] == c.mpr_seed + 1
    assert gathered[0][3] != gathered[1][3]
    assert sharding.throughput(units_total, ms_max) == units_total / 0.015


def test_single_rank_needs_no_process_group():
    assert not dist.is_initialized()
    assert sharding.aggregate(3.5, 7.0, 9, 1) == (3.5, 7.0, 9)


def test_multi_rank_without_group_fails_loudly():
    with pytest.raises(RuntimeError):
        sharding.aggregate(1.0, 1.0, 1, 2)


def test_rank_problem_rejects_bad_rank():
    with pytest.raises(ValueError):
        sharding.rank_problem(0, 0, 2, 2)
    with pytest.raises(ValueError):
        sharding.throughput(1.0, 0.0)
