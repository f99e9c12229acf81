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


@pytest.mark.parametrize("seed", [21, 22])
def test_random_dp_configurations_match_the_oracle(oracle_mod, seed):
    """The same idea against the oracle: DP on random shapes, masked fractions, temperatures, schedules, quench counts and
    q in (0, 1/2], on a random path -- identical accepted-move counts, spins to 1e-9, energies to 1e-10, predictions to
    1e-9 of the data range."""
    import torch
    from paper_1910_08448_b200 import mpr
    rng = np.random.default_rng(seed)
    done = 0
    while done < 40:
        Ly, Lx = int(rng.integers(1, 140)), int(rng.integers(1, 140))
        if min(Ly, Lx) < 2:          # single rows / columns: see test_over_relaxation_tie_at_the_edge_of_the_range
            continue
        f = float(rng.choice([0.05, 0.33, 0.66, 0.9, 0.99]))
        values = rng.normal(50, 10, (Ly, Lx))
        mask = (rng.uniform(size=(Ly, Lx)) < f).astype(np.uint8)
        if int((mask == 0).sum()) < 2:
            mask.reshape(-1)[:2] = 0
        values[mask == 1] = np.nan
        sched = str(rng.choice(["R4", "SITE_FUSED"]))
        T = float(10 ** rng.uniform(-3.0, 0.5))
        q = float(rng.choice([0.5, 0.5, 0.5, 0.37, 0.2]))
        chain_seed, nq = int(rng.integers(0, 2 ** 40)), int(rng.choice([0, 1, 4, 32]))
        n_sw, n_me = int(rng.integers(1, 7)), int(rng.integers(1, 4))
        path = str(rng.choice(["AUTO", "PLAIN", "LIST", "STRIP"] + (["TILED"] if sched == "R4" else [])))
        what = ((Ly, Lx), f, sched, T, q, chain_seed, nq, n_sw, n_me, path)
        o = oracle_mod.Oracle(values=values, mask=mask, seed=chain_seed)
        g = mpr.Mpr(values, mask, mode="DP", seed=chain_seed)
        for h in (o, g):
            h.set_quench(nq)
            if q != 0.5:
                h.set_q(q)
            h.set_schedule(sched)
            h.set_temperature(T)
        g.set_path(path)
        pred_o, e_o, se_o = o.run(n_sw, n_me)
        pred_g, e_g, se_g = g.run(n_sw, n_me)
        assert g.counters() == o.counters(), what
        assert np.max(np.abs(g.get_state().cpu().numpy() - o.get_state())) <= 1e-9, what
        assert abs(e_g - e_o) <= 1e-10 and abs(se_g - se_o) <= 1e-10, what
        zr = o.zrange()
        assert np.max(np.abs(np.nan_to_num(pred_g.cpu().numpy() - pred_o))) <= 1e-9 * (zr[1] - zr[0]), what
        g.close()
        done += 1
