"""Host logic of the slab decomposition (paper_1910_08448_b200/slabs.py) on CPU: the partition, which rows
travel and how often, the lock step of sweeps, exchanges and measurements, the reductions, the temperature matching over
slabs -- driven with tests/helpers/toy_slab.py (an integer automaton with the dependency structure of the MPR sweep and
none of its arithmetic) in one process and as two real processes over gloo on 127.0.0.1 (DistTransport: send / recv of
the halo rows, all_reduce of the energies).  A slab run must reproduce the whole-grid run exactly.  No GPU."""
import os
import socket
import sys

import numpy as np
import pytest
import torch.distributed as dist
import torch.multiprocessing as mp

sys.path.insert(0, os.path.join(os.path.dirname(os.path.abspath(__file__)), "helpers"))
from toy_slab import ToySlab  # noqa: E402

from paper_1910_08448_b200 import mpr, slabs  # noqa: E402  (host-only routines of the library; no GPU call)


def problem(Ly=64, Lx=37, seed=3, f=0.7):
    rng = np.random.default_rng(seed)
    values = rng.normal(50.0, 10.0, (Ly, Lx))
    mask = (rng.uniform(size=(Ly, Lx)) < f).astype(np.uint8)
    values[mask == 1] = np.nan
    return values, mask


def build(values, mask, count, halo, transport=None, n_quench=6):
    plans = slabs.plan_slabs(mask.shape[0], count, halo)
    transport = transport or slabs.LocalTransport()
    mine = [p for p in plans if transport.owner(p.index) == transport.rank]
    objs = {p.index: ToySlab(p, values, mask, seed=21) for p in mine}
    return slabs.SlabSet(plans, objs, mask.shape[1], transport, n_quench=n_quench, trial_lengths=(9, 20),
                         stats=mpr.debug_series_stats, match=mpr.debug_match_temperature)


def run_all(ss):
    T_hat = ss.estimate_temperature()
    series, e, se = ss.run(7, 21)
    return dict(T=T_hat, trials=ss.n_trials, series=series, e=e, se=se, state=ss.state(), pred=ss.prediction(),
                acc=ss.accepted(), e_sample=ss.e_sample, n_pairs=ss.n_pairs, n_free=ss.n_free, zr=(ss.z_min, ss.z_max),
                exchanges=ss.exchanges)


def same(a, b):
    assert np.array_equal(a["state"], b["state"]) and np.array_equal(a["pred"], b["pred"])
    assert a["acc"] == b["acc"] and a["n_pairs"] == b["n_pairs"] and a["n_free"] == b["n_free"] and a["zr"] == b["zr"]
    assert a["trials"] == b["trials"]
    assert abs(a["T"] - b["T"]) <= 1e-12 * a["T"] and abs(a["e_sample"] - b["e_sample"]) <= 1e-15
    assert np.max(np.abs(a["series"] - b["series"])) <= 1e-13 and abs(a["e"] - b["e"]) <= 1e-13


@pytest.mark.parametrize("count,halo", [(2, 4), (2, 8), (3, 8), (4, 12), (5, 4)])
def test_slabs_reproduce_the_whole_grid(count, halo):
    values, mask = problem()
    ref = run_all(build(values, mask, 1, 8))
    assert ref["exchanges"] == 0 and 0.15 < ref["T"] < 0.25       # the toy's e(T) = -2 + T crosses e_sample = -1.8 there
    got = run_all(build(values, mask, count, halo))
    same(ref, got)
    assert got["exchanges"] > 0


def test_a_late_exchange_is_caught():
    """The test above has teeth: with exchanges every halo / 4 + 1 sweeps instead of halo / 4 the spoiled rows reach the
    owned ones and the result differs."""
    values, mask = problem()
    ref = build(values, mask, 1, 4)
    bad = build(values, mask, 3, 4)
    for ss in (ref, bad):
        ss.set_temperature(0.2)
        ss.reset_chain(0)
    ref.sweep(6)
    bad.sweeps_per_exchange = 2       # pretends the halo lasts two sweeps; it holds 4 rows
    bad.sweep(6)
    assert not np.array_equal(ref.state(), bad.state())


def test_moves_cover_exactly_the_halos():
    plans = slabs.plan_slabs(100, 3, 8)
    values, mask = problem(100, 10)
    ss = build(values, mask, 3, 8)
    filled = {p.index: set() for p in plans}
    for (src, src_row, dst, dst_row, n) in ss.moves():
        ps, pd = plans[src], plans[dst]
        assert ps.own_begin <= src_row and src_row + n <= ps.own_end          # only owned rows are sent
        assert ps.row0_g + src_row == pd.row0_g + dst_row                     # to the same global rows
        filled[dst] |= set(range(dst_row, dst_row + n))
    for p in plans:
        halo_rows = set(range(0, p.own_begin)) | set(range(p.own_end, p.n_rows))
        assert filled[p.index] == halo_rows


def _free_port():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def _worker(rank, world, port, out):
    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    try:
        values, mask = problem()
        ss = build(values, mask, world, 8, transport=slabs.DistTransport())
        assert list(ss.slabs) == [rank]                                        # one slab per rank
        res = run_all(ss)
        out[rank] = res
    finally:
        dist.destroy_process_group()


@pytest.mark.timeout(300)
def test_two_ranks_over_gloo():
    world, port = 2, _free_port()
    with mp.Manager() as mgr:
        out = mgr.dict()
        mp.spawn(_worker, args=(world, port, out), nprocs=world, join=True)
        res = dict(out)
    assert set(res) == {0, 1}
    values, mask = problem()
    ref = run_all(build(values, mask, 1, 8))
    for r in (0, 1):                     # every rank ends with the whole result, equal to the single-process one
        same(ref, res[r])
