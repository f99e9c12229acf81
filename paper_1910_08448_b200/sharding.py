"""Host-side sharding of the MPR path over ranks.

The path shards by INDEPENDENT PROBLEMS (the paper's M realisations of the sampling mask,
PAPER.md:57): every rank runs the whole hot path on its own field / mask / chain seed and there
is no data-path collective.  The only exchange is the measurement itself: the timed region's
duration is the MAX over ranks, the processed units and launch counts are SUMS over ranks.

This module holds no arithmetic of the method and touches no kernel; `bench.py` uses it on NCCL,
`tests/test_sharding_gloo.py` on gloo with world_size 2.
"""
from dataclasses import dataclass

import torch
import torch.distributed as dist

# rank r takes field seed + FIELD_SEED_STRIDE * r and chain seed + r: rank 0 is BASELINE.json's
# configuration unchanged, and no two ranks share a field, a mask or a Philox key.
FIELD_SEED_STRIDE = 1000


@dataclass(frozen=True)
class RankProblem:
    rank: int
    world: int
    field_seed: int
    mpr_seed: int


def rank_problem(field_seed: int, mpr_seed: int, rank: int, world: int) -> RankProblem:
    """Seeds of the problem rank `rank` of `world` works on (weak scaling: same recipe and size)."""
    if world < 1 or not (0 <= rank < world):
        raise ValueError("rank %d outside world of size %d" % (rank, world))
    return RankProblem(rank, world, field_seed + FIELD_SEED_STRIDE * rank, mpr_seed + rank)


def aggregate(ms: float, units: float, launches: int, world: int, device="cpu"):
    """(max over ranks of ms, sum of units, sum of launches) -- every rank gets the same triple.

    With world == 1 no process group is needed.  `device` is where the reduction tensors live
    (the rank's GPU under NCCL, "cpu" under gloo).
    """
    if world == 1:
        return float(ms), float(units), int(launches)
    if not dist.is_initialized():
        raise RuntimeError("aggregate(world=%d) needs an initialised process group" % world)
    t = torch.tensor([float(ms)], dtype=torch.float64, device=device)
    s = torch.tensor([float(units), float(launches)], dtype=torch.float64, device=device)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    dist.all_reduce(s, op=dist.ReduceOp.SUM)
    return float(t.item()), float(s[0].item()), int(round(float(s[1].item())))


def throughput(units_total: float, ms_max: float) -> float:
    """Whole-job units per second: all ranks' units over the slowest rank's device time."""
    if ms_max <= 0.0:
        raise ValueError("non-positive duration")
    return units_total / (ms_max * 1e-3)
