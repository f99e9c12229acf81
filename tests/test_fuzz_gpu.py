"""Differential fuzzing on the GPU, fixed seed: random shapes (1 .. 400 rows and columns, square or not), masked fractions,
precision modes, schedules, temperatures, quench counts and sweep counts; every kernel path (STRIP at depth 1 and 2, LIST,
TILED at depth 1 .. 4, AUTO with the library's own choices) and the slab decomposition (copies and peer stores) must give
the spins, accepted-move counts and predictions of the per-pass PLAIN kernels, bit for bit.  (PLAIN itself is tied to the
oracle by the DP parity tests.)  An unbounded version of this loop found the one defect fixed by mpr_create_slab."""
import numpy as np
import pytest

pytestmark = pytest.mark.gpu

MODES = ["DP", "SP", "SP_PRECISE", "SP_INTRINSIC", "DS_INTRINSIC", "HP"]


@pytest.mark.parametrize("seed", [11, 12, 13])
def test_random_configurations_agree_with_the_per_pass_kernels(seed):
    import torch
    assert torch.cuda.is_available(), "GPU tests need a CUDA device"
    from paper_1910_08448_b200 import build, mpr, slabs
    build.build()
    rng = np.random.default_rng(seed)
    done = 0
    while done < 200:
        Ly, Lx = int(rng.integers(1, 400)), int(rng.integers(1, 400))
        if rng.uniform() < 0.3:
            Ly = Lx
        if Ly * Lx < 2:
            continue
        f = float(rng.choice([0.05, 0.33, 0.66, 0.9, 0.99]))
        values = rng.normal(50, 10, (Ly, Lx))
        mask = (rng.uniform(size=(Ly, Lx)) < f).astype(np.uint8)
        if int((mask == 0).sum()) < 2:
            mask.reshape(-1)[:2] = 0
        values[mask == 1] = np.nan
        mode, sched = str(rng.choice(MODES)), str(rng.choice(["R4", "SITE_FUSED"]))
        T = float(10 ** rng.uniform(-3.5, 0.5))
        chain_seed, nq = int(rng.integers(0, 2 ** 40)), int(rng.choice([0, 1, 2, 5, 32]))
        n_sw, n_me = int(rng.integers(1, 8)), int(rng.integers(0, 4))
        what = ((Ly, Lx), f, mode, sched, T, chain_seed, nq, n_sw, n_me)

        def run(path, k):
            g = mpr.Mpr(values, mask, mode=mode, seed=chain_seed)
            g.set_path(path); g.set_fused_sweeps(k); g.set_schedule(sched); g.set_quench(nq); g.set_temperature(T)
            pred, e, se = g.run(n_sw, n_me)
            out = (g.get_state().cpu(), g.counters(), torch.nan_to_num(pred.cpu(), nan=-1.0), e)
            g.close()
            return out

        ref = run("PLAIN", 1)
        cases = [("STRIP", 1), ("STRIP", 2), ("LIST", 1), ("AUTO", 0)]
        if sched == "R4":
            cases += [("TILED", 1), ("TILED", int(rng.integers(2, 5)))]
        for path, k in cases:
            got = run(path, k)
            assert torch.equal(got[0], ref[0]) and got[1] == ref[1] and torch.equal(got[2], ref[2]), (what, path, k)
            assert n_me == 0 or abs(got[3] - ref[3]) <= 3e-6 * abs(ref[3]) + 1e-12, (what, path, k)
        if Ly >= 40 and nq % 2 == 0 and mode in ("DP", "SP", "SP_INTRINSIC", "HP"):
            count = int(rng.integers(2, 4))
            for peer in (False, True):
                ss = slabs.make_slab_set(values, mask, count, halo=4 if peer else int(rng.choice([4, 8])), mode=mode,
                                         seed=chain_seed, path="STRIP", schedule=sched, n_quench=nq, peer=peer)
                ss.set_temperature(T)
                ss.reset_chain(0)
                ss.run(n_sw, n_me)
                assert np.array_equal(ss.state(), ref[0].numpy()) and ss.accepted() == ref[1][0], (what, count, peer)
                assert np.array_equal(np.nan_to_num(ss.prediction(), nan=-1.0), ref[2].numpy()), (what, count, peer)
        done += 1
