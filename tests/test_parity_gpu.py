"""Parity of the CUDA path (through the C ABI, paper_1910_08448_b200.mpr) with the CPU oracle on the
same seeded inputs.  Gates (BASELINE.json north_star): DP makes identical accept/reject decisions
and |dphi| <= 1e-9 per site after 10 sweeps; integer counters bit-exact; both kernel paths and
every fused depth give bit-identical spins; SP modes are judged statistically."""
import math

import numpy as np
import pytest

pytestmark = pytest.mark.gpu

TWO_PI = 2.0 * math.pi
PHI_TOL = 1e-9      # north_star: per-site |dphi| <= 1e-9 after 10 sweeps (DP)


@pytest.fixture(scope="module")
def mpr():
    import torch
    assert torch.cuda.is_available(), "GPU tests need a CUDA device"
    from paper_1910_08448_b200 import build, mpr as m
    build.build()
    m.lib()
    return m


@pytest.fixture(scope="module")
def inputs():
    from paper_1910_08448_b200 import inputs as i
    return i


def phi_diff(a, b):
    return float(np.max(np.abs(np.asarray(a) - np.asarray(b))))


def make(inputs, L, xi, seed, f, lognormal=False):
    return inputs.make_problem(L, xi, seed, f, lognormal)


# --------------------------------------------------------------------------- generator
def test_device_philox_matches_oracle(mpr, oracle_mod):
    rng = np.random.default_rng(7)
    ctr = rng.integers(0, 2 ** 32, (4096, 4), dtype=np.uint64).astype(np.uint32)
    ctr[0] = 0
    ctr[1] = 0xFFFFFFFF
    key = (0x12345678, 0x9ABCDEF0)
    out = mpr.debug_philox(ctr, key)
    for i in range(0, 4096, 37):
        assert list(out[i]) == oracle_mod.philox4x32_10(list(ctr[i]), key), i


# --------------------------------------------------------------------------- set-up (R1, R6)
@pytest.mark.parametrize("L,xi,f", [(64, 8.0, 0.33), (100, 10.0, 0.66), (131, 9.0, 0.9)])
def test_setup_matches_oracle(mpr, oracle_mod, inputs, L, xi, f):
    values, mask, _ = make(inputs, L, xi, 5, f)
    g = mpr.Mpr(values, mask, seed=11)
    o = oracle_mod.Oracle(values=values, mask=mask, seed=11)
    info = g.info()
    assert (info["z_min"], info["z_max"]) == o.zrange()
    assert info["n_free"] == int(mask.sum())
    es_g, n_g = g.sample_energy()
    es_o, n_o = o.sample_energy()
    assert n_g == n_o
    assert abs(es_g - es_o) <= 1e-12 * abs(es_o)
    # R8 initial state: uniform spins + 32 quench double passes
    assert phi_diff(g.get_state().cpu().numpy(), o.get_state()) <= PHI_TOL
    H_g, e_g = g.energy()
    H_o, e_o = o.energy()
    assert abs(H_g - H_o) <= 1e-11 * abs(H_o)
    assert abs(e_g - e_o) <= 1e-12 * abs(e_o)


def test_error_paths(mpr, inputs):
    L = 16
    rng = np.random.default_rng(1)
    z = rng.normal(50, 10, (L, L))
    mask = (rng.uniform(size=(L, L)) < 0.5).astype(np.uint8)
    for vals, msk, code in [
        (z, np.ones((L, L), dtype=np.uint8), mpr.ERR_NO_MEASURED),
        (np.full((L, L), 3.0), np.zeros((L, L), dtype=np.uint8), mpr.ERR_DEGENERATE_RANGE),
        (np.where(mask == 1, 1.0, np.inf), mask, mpr.ERR_NONFINITE),
    ]:
        with pytest.raises(mpr.MprError) as ei:
            mpr.Mpr(vals, msk)
        assert ei.value.code == code
    vals = z.copy()
    vals[mask == 1] = np.nan                     # values at prediction sites are never read
    g = mpr.Mpr(vals, mask)
    with pytest.raises(mpr.MprError) as ei:
        g.run(1, 1)
    assert ei.value.code == mpr.ERR_NOT_READY
    with pytest.raises(mpr.MprError) as ei:
        g.set_temperature(0.0)
    assert ei.value.code == mpr.ERR_INVALID_ARG
    with pytest.raises(mpr.MprError):
        g.set_fused_sweeps(5)
    g.set_fused_sweeps(0)                        # 0 = the library's choice


# --------------------------------------------------------------------------- DP parity, pass by pass
@pytest.mark.parametrize("path", ["PLAIN", "TILED", "STRIP"])
@pytest.mark.parametrize("L,xi,f,T", [(64, 8.0, 0.33, 0.07), (97, 8.0, 0.9, 0.02), (250, 16.0, 0.66, 0.3)])
def test_dp_ten_sweeps_match_oracle(mpr, oracle_mod, inputs, L, xi, f, T, path):
    values, mask, _ = make(inputs, L, xi, 3, f)
    g = mpr.Mpr(values, mask, seed=1000)
    o = oracle_mod.Oracle(values=values, mask=mask, seed=1000)
    g.set_temperature(T)
    o.set_temperature(T)
    g.set_path(path)
    g.sweep(10)
    o.hybrid_sweeps(10)
    sg, so = g.get_state().cpu().numpy(), o.get_state()
    assert phi_diff(sg, so) <= PHI_TOL
    acc_g, att_g, sw_g = g.counters()
    acc_o, att_o, sw_o = o.counters()
    assert (acc_g, att_g, sw_g) == (acc_o, att_o, sw_o)      # identical accept/reject decisions
    assert sg.min() >= 0.0 and sg.max() <= TWO_PI + 1e-15
    # measured spins never move
    m0 = mask == 0
    assert np.array_equal(sg[m0], g.get_state().cpu().numpy()[m0])
    assert phi_diff(sg[m0], so[m0]) <= 1e-12


def test_dp_single_passes_match_oracle(mpr, oracle_mod, inputs):
    """Each kind of colour pass alone, including edge and corner sites (open boundaries, R2)."""
    L = 33
    values, mask, _ = make(inputs, L, 5.0, 9, 0.8)
    g = mpr.Mpr(values, mask, seed=5)
    o = oracle_mod.Oracle(values=values, mask=mask, seed=5)
    g.set_quench(0)
    o.set_quench(0)
    g.set_temperature(0.5)
    o.set_temperature(0.5)
    assert phi_diff(g.get_state().cpu().numpy(), o.get_state()) <= 1e-12      # uniform init (R8)
    for step, (kind, c) in enumerate([("MET", 0), ("MET", 1), ("OR", 0), ("OR", 1), ("QUENCH", 1), ("QUENCH", 0),
                                      ("MET", 1), ("OR", 0)]):
        g.pass_(kind, c, sweep=step + 1)
        if kind == "MET":
            o.met_pass(c, step + 1)
        elif kind == "OR":
            o.or_pass(c)
        else:
            o.quench_pass(c)
        assert phi_diff(g.get_state().cpu().numpy(), o.get_state()) <= PHI_TOL, (step, kind, c)
    assert g.counters()[0] == o.counters()[0]


@pytest.mark.parametrize("L", [2, 3, 5, 16])
def test_tiny_grids(mpr, oracle_mod, L):
    rng = np.random.default_rng(L)
    z = rng.normal(50, 10, (L, L))
    mask = np.zeros((L, L), dtype=np.uint8)
    mask.flat[rng.choice(L * L, size=max(1, L * L // 2), replace=False)] = 1
    mask[0, 0] = 0
    mask[-1, -1] = 0
    g = mpr.Mpr(z, mask, seed=3)
    o = oracle_mod.Oracle(values=z, mask=mask, seed=3)
    for path in ("PLAIN", "TILED", "STRIP"):
        g.set_path(path)
        g.set_seed(3)
        o.set_seed(3)
        g.set_temperature(0.2)
        o.set_temperature(0.2)
        g.sweep(10)
        o.hybrid_sweeps(10)
        assert phi_diff(g.get_state().cpu().numpy(), o.get_state()) <= PHI_TOL
        assert g.counters() == o.counters()


# --------------------------------------------------------------------------- whole run (R15, R3)
def test_dp_run_matches_oracle_config1(mpr, oracle_mod, inputs):
    """BASELINE.json configs[0]: L = 64, 33 % masked, 100 + 100 sweeps, DP."""
    c, values, mask, truth = inputs.make_config(1)
    g = mpr.Mpr(values, mask, seed=c.mpr_seed)
    o = oracle_mod.Oracle(values=values, mask=mask, seed=c.mpr_seed)
    g.set_temperature(0.07)
    o.set_temperature(0.07)
    pred_g, e_g, se_g = g.run(c.n_eq, c.n_meas)
    pred_o, e_o, se_o = o.run(c.n_eq, c.n_meas)
    pred_g = pred_g.cpu().numpy()
    m1 = mask == 1
    assert np.array_equal(pred_g[~m1], values[~m1])                 # measured sites bit-exact
    zmin, zmax = o.zrange()
    assert np.max(np.abs(pred_g[m1] - pred_o[m1])) <= 1e-8 * (zmax - zmin)
    assert abs(e_g - e_o) <= 1e-11 and abs(se_g - se_o) <= 1e-11
    np.testing.assert_allclose(g.series(), o.series(), rtol=0, atol=1e-11)
    assert g.counters() == o.counters()
    mae_g, rmse_g = inputs.prediction_errors(pred_g, truth, mask)
    mae_o, rmse_o = inputs.prediction_errors(pred_o, truth, mask)
    assert abs(mae_g - mae_o) <= 1e-8 and abs(rmse_g - rmse_o) <= 1e-8
    # chain continuation: a second run averages over all 200 measurement sweeps
    pred_g2, _, _ = g.run(0, c.n_meas)
    pred_o2, _, _ = o.run(0, c.n_meas)
    assert np.max(np.abs(pred_g2.cpu().numpy()[m1] - pred_o2[m1])) <= 1e-8 * (zmax - zmin)


def test_temperature_estimate_matches_oracle(mpr, oracle_mod, inputs):
    c, values, mask, _ = inputs.make_config(1)
    g = mpr.Mpr(values, mask, seed=c.mpr_seed)
    o = oracle_mod.Oracle(values=values, mask=mask, seed=c.mpr_seed)
    T_g, es_g, n_g = g.estimate_temperature()
    T_o, es_o, n_o = o.estimate_temperature()
    assert abs(es_g - es_o) <= 1e-12
    assert n_g == n_o
    assert abs(T_g - T_o) <= 1e-9 * T_o
    # the chain was reset (trial 0) with T set: the next sweeps agree as well
    g.sweep(3)
    o.hybrid_sweeps(3)
    assert phi_diff(g.get_state().cpu().numpy(), o.get_state()) <= PHI_TOL


def test_no_root_is_reported(mpr):
    L = 12
    z = np.where(np.arange(L)[None, :] < 6, 10.0, 20.0) * np.ones((L, 1))
    rng = np.random.default_rng(0)
    mask = np.zeros((L, L), dtype=np.uint8)
    mask[:, 5:7] = 1
    mask[rng.integers(0, L, 20), rng.integers(0, 4, 20)] = 1
    g = mpr.Mpr(z, mask, seed=2)
    assert g.sample_energy()[0] == -2.0
    with pytest.raises(mpr.MprError) as ei:
        g.estimate_temperature()
    assert ei.value.code == mpr.ERR_NO_ROOT


def test_run_timing_reports_the_equilibration_launches(mpr, inputs):
    """mpr_get_run_timing: device time, launches and sweeps of the equilibration phase of the last run
    (what bench.py divides to get the dominant kernel's average duration inside the timed step)."""
    values, mask, _ = make(inputs, 300, 12.0, 4, 0.66)
    g = mpr.Mpr(values, mask, mode="SP_INTRINSIC", seed=5)
    g.set_temperature(0.05)
    with pytest.raises(mpr.MprError) as ei:
        g.run_timing()
    assert ei.value.code == mpr.ERR_NOT_READY
    g.set_path("TILED")
    g.run(20, 3)
    ms, launches, sweeps = g.run_timing()
    assert (launches, sweeps) == (5, 20) and 0.0 < ms < 1000.0        # the library's choice at L = 300: 4 sweeps per launch
    g.set_fused_sweeps(1)
    g.run(20, 3)
    assert g.run_timing()[1:] == (20, 20)                               # tiled, one sweep per launch
    g.set_fused_sweeps(4)
    g.run(18, 2)
    ms4, launches4, sweeps4 = g.run_timing()
    assert (launches4, sweeps4) == (5, 18) and ms4 > 0.0                # 4 + 4 + 4 + 4 + 2
    g.run(0, 2)
    assert g.run_timing() == (0.0, 0, 0)
    g.set_path("PLAIN")
    g.run(3, 1)
    assert g.run_timing()[1:] == (12, 3)                                # one launch per colour pass
    g.set_path("STRIP")
    g.run(9, 1)
    assert g.run_timing()[1:] == (5, 9)                                 # 2 + 2 + 2 + 2 + 1 at depth min(4, 2)
    g.close()


# --------------------------------------------------------------------------- determinism contract
@pytest.mark.parametrize("mode", ["DP", "SP", "SP_PRECISE", "SP_INTRINSIC"])
def test_paths_and_fused_depths_are_bit_identical(mpr, inputs, mode):
    L = 300                                  # several tiles in x and y, ragged in both
    values, mask, _ = make(inputs, L, 12.0, 4, 0.66)
    g = mpr.Mpr(values, mask, mode=mode, seed=77)
    g.set_temperature(0.05)
    ref = None
    for path, k in [("PLAIN", 1), ("TILED", 1), ("TILED", 2), ("TILED", 3), ("TILED", 4), ("STRIP", 1), ("STRIP", 2)]:
        g.set_path(path)
        g.set_fused_sweeps(k)
        g.reset_chain(0)
        g.sweep(9)                            # 9 is not a multiple of 2 or 4: ragged last launch
        st = g.get_state().cpu().numpy()
        cnt = g.counters()
        if ref is None:
            ref = (st, cnt)
        else:
            assert np.array_equal(st, ref[0]), (path, k)
            assert cnt == ref[1], (path, k)
    # measurement launches: energies and accumulators agree between the paths
    out = []
    for path in ("PLAIN", "TILED", "STRIP"):
        g.set_path(path)
        g.reset_chain(0)
        pred, e, se = g.run(5, 7)
        out.append((pred.cpu().numpy(), g.series()))
    for other in out[1:]:
        assert np.array_equal(out[0][0], other[0])
        np.testing.assert_allclose(out[0][1], other[1], rtol=0, atol=1e-13)
    # the site-fused schedule (R4b): STRIP at both depths equals the plain per-pass kernels
    g.set_schedule("SITE_FUSED")
    ref = None
    for path, k in [("PLAIN", 1), ("STRIP", 1), ("STRIP", 2)]:
        g.set_path(path)
        g.set_fused_sweeps(k)
        g.reset_chain(0)
        g.sweep(7)
        pred, e, se = g.run(2, 3)
        cur = (g.get_state().cpu().numpy(), g.counters(), pred.cpu().numpy(), g.series())
        if ref is None:
            ref = cur
        else:
            assert np.array_equal(cur[0], ref[0]) and cur[1] == ref[1], (path, k)
            assert np.array_equal(cur[2], ref[2]), (path, k)
            np.testing.assert_allclose(cur[3], ref[3], rtol=0, atol=1e-13)


@pytest.mark.parametrize("mode", ["DP", "SP", "SP_PRECISE", "SP_INTRINSIC"])
def test_pass_synchronisation_stress(mpr, inputs, mode):
    """DP, SP and SP_PRECISE separate the colour passes of a tile by pairwise named barriers between
    neighbouring warps instead of a CTA-wide barrier (mpr_tiled.cuh, neighbour_sync).  A missing or
    misplaced synchronisation shows up as a spin that differs from the one-launch-per-pass PLAIN
    path, most likely where the warps of a CTA can drift furthest apart: the deepest fusion (k = 4,
    16 passes per launch) on a grid of many tiles, repeated.  compute-sanitizer's racecheck is not
    available on the GPU pool, so this bitwise comparison is the check that stands in for it; it
    is evidence, not a proof of race freedom."""
    import torch
    L = 2048
    values, mask, _ = make(inputs, L, 48.0, 9, 0.9)
    dv, dm = torch.from_numpy(values).cuda(), torch.from_numpy(mask).cuda()
    out = {}
    for path, k in (("PLAIN", 1), ("TILED", 4), ("TILED", 1), ("STRIP", 2), ("STRIP", 1)):
        g = mpr.Mpr(dv, dm, mode=mode, seed=4242)
        g.set_path(path)
        g.set_fused_sweeps(k)
        g.set_temperature(0.02)
        states = []
        for _ in range(3):                    # 3 x 8 sweeps: six launches of 16 passes at k = 4
            g.sweep(8)
            states.append(g.get_state())
        out[(path, k)] = (states, g.counters())
        g.close()
    ref_states, ref_cnt = out[("PLAIN", 1)]
    for key in (("TILED", 4), ("TILED", 1), ("STRIP", 2), ("STRIP", 1)):
        states, cnt = out[key]
        assert cnt == ref_cnt, (mode, key, cnt, ref_cnt)
        for i, (a, b) in enumerate(zip(states, ref_states)):
            assert torch.equal(a, b), (mode, key, i, int((a != b).sum()))


# --------------------------------------------------------------------------- SP modes: statistics
def test_sp_modes_statistics_config2_shape(mpr, oracle_mod, inputs):
    """e within 3 standard errors of the DP value; MAE / RMSE within 1 % of the DP oracle's."""
    L = 256
    values, mask, truth = make(inputs, L, 16.0, 1, 0.66)
    T = 0.03
    o = oracle_mod.Oracle(values=values, mask=mask, seed=1001, threads=oracle_mod.threads_available())
    o.set_temperature(T)
    pred_o, e_o, se_o = o.run(300, 200)
    mae_o, rmse_o = inputs.prediction_errors(pred_o, truth, mask)
    for mode in ("DP", "SP", "SP_PRECISE", "SP_INTRINSIC"):
        es, maes = [], []
        for seed in (1001, 2002, 3003, 4004):
            g = mpr.Mpr(values, mask, mode=mode, seed=seed)
            g.set_temperature(T)
            pred, e, se = g.run(300, 200)
            es.append(e)
            mae, rmse = inputs.prediction_errors(pred.cpu().numpy(), truth, mask)
            maes.append((mae, rmse))
        e_mean = float(np.mean(es))
        e_se = float(np.std(es, ddof=1) / math.sqrt(len(es)))
        assert abs(e_mean - e_o) <= 3.0 * math.hypot(e_se, se_o) + 1e-6, (mode, e_mean, e_o, e_se, se_o)
        mae = float(np.mean([m for m, _ in maes]))
        rmse = float(np.mean([r for _, r in maes]))
        assert abs(mae / mae_o - 1.0) <= 0.01, (mode, mae, mae_o)
        assert abs(rmse / rmse_o - 1.0) <= 0.01, (mode, rmse, rmse_o)


@pytest.mark.parametrize("lognormal,f,T", [(False, 0.9, 1.1e-3), (True, 0.33, 1.5e-3)])
def test_float_modes_at_low_temperature(mpr, inputs, lognormal, f, T):
    """The low-T stress point (T_hat ~ 1e-3 at configs 3 and 5; lognormal = spins crowded
    near phi = 0).  Two separate statements about the float modes, on chain snapshots whose energy is
    evaluated twice -- by the mode's own S5 arithmetic and by a DP context loaded with the same phi:

    (a) evaluation: the mode's own e of a state equals the DP evaluation of that state to 5e-10.  With
        u.F in float arithmetic this was a constant +1e-8 .. +2.6e-8, ~3 standard errors of e at
        L = 16384 (u_s.u_t is sensitive to the norm error of the stored float vectors and to the
        rounding of a value near 1; which of the two dominated was not separated); the per-bond form
        1 - |u_s - u_t|^2 / 2 (site_energy_term), sensitive to neither, brings it to ~1e-11.
    (b) chain: the DP-evaluated mean e of each mode's chain is within 3 standard errors of the DP
        chain's (north_star's statistical gate).  The reference is the GPU DP chain, which the tests
        above show to be decision-identical to the oracle; seeds are fixed, so the outcome is
        reproducible rather than a draw."""
    # 10 seeds: the standard error of a mode's mean is itself estimated from the seeds, and with 3 of them (2 degrees of
    # freedom) a "3 standard errors" gate fails one time in eleven by chance alone
    L, n_eq, n_snap, gap, seeds = 2048, 400, 12, 25, tuple(range(11, 111, 10))
    values, mask, _ = make(inputs, L, 64.0, 4, f, lognormal)
    import torch
    dv, dm = torch.from_numpy(values).cuda(), torch.from_numpy(mask).cuda()
    ev = mpr.Mpr(dv, dm, mode="DP", seed=1)
    ev.set_temperature(T)
    stats = {}
    for mode in ("DP", "SP", "SP_PRECISE", "SP_INTRINSIC"):
        per_seed, worst_eval = [], 0.0
        for seed in seeds:
            g = mpr.Mpr(dv, dm, mode=mode, seed=seed)
            g.set_temperature(T)
            g.sweep(n_eq)
            dp = []
            for _ in range(n_snap):
                g.sweep(gap)
                own = g.energy()[1]
                ev.set_state(g.get_state())
                e_dp = ev.energy()[1]
                worst_eval = max(worst_eval, abs(own - e_dp))
                dp.append(e_dp)
            per_seed.append(float(np.mean(dp)))
            g.close()
        stats[mode] = (float(np.mean(per_seed)), float(np.std(per_seed, ddof=1) / math.sqrt(len(seeds))), worst_eval)
    ev.close()
    e_ref, se_ref, _ = stats["DP"]
    assert -2.0 < e_ref < -1.99                                   # a low-temperature state, not a frozen one
    for mode in ("SP", "SP_PRECISE", "SP_INTRINSIC"):
        e_m, se_m, worst_eval = stats[mode]
        assert worst_eval <= 5e-10, (mode, worst_eval)                                   # (a)
        assert abs(e_m - e_ref) <= 3.0 * math.hypot(se_m, se_ref), (mode, e_m, e_ref, se_m, se_ref)   # (b)


# --------------------------------------------------------------------------- BASELINE configs at their actual sizes
def _float_mode_gates(mpr, inputs, dv, dm, truth, mask, modes, seed, T, n_eq, n_meas, e_o, se_o, mae_o, rmse_o):
    """north_star's statistical gates for the float modes against the DP oracle run (e_o, se_o, mae_o, rmse_o)."""
    for mode in modes:
        g = mpr.Mpr(dv, dm, mode=mode, seed=seed)
        g.set_temperature(T)
        pred, e, se = g.run(n_eq, n_meas)
        mae, rmse = inputs.prediction_errors(pred.cpu().numpy(), truth, mask)
        g.close()
        assert abs(e - e_o) <= 3.0 * math.hypot(se, se_o), (mode, e, e_o, se, se_o)
        assert abs(mae / mae_o - 1.0) <= 0.01, (mode, mae, mae_o)
        assert abs(rmse / rmse_o - 1.0) <= 0.01, (mode, rmse, rmse_o)


def test_config2_actual_size(mpr, oracle_mod, inputs):
    """BASELINE.json configs[1] as stated: L = 512, 66 % masked, temperature inferred by energy matching,
    1000 + 100 sweeps, DP versus SP storage.  DP: the whole procedure (T-matching trials, run) equals the
    oracle's -- same T_hat, same accepted-move count, same prediction; SP: the statistical gates."""
    import torch
    c, values, mask, truth = inputs.make_config(2)
    dv, dm = torch.from_numpy(values).cuda(), torch.from_numpy(mask).cuda()
    o = oracle_mod.Oracle(values=values, mask=mask, seed=c.mpr_seed, threads=oracle_mod.threads_available())
    g = mpr.Mpr(dv, dm, seed=c.mpr_seed)
    T_o, es_o, n_o = o.estimate_temperature()
    T_g, es_g, n_g = g.estimate_temperature()
    assert n_g == n_o and abs(es_g - es_o) <= 1e-12 and abs(T_g - T_o) <= 1e-9 * T_o
    pred_o, e_o, se_o = o.run(c.n_eq, c.n_meas)
    pred_g, e_g, se_g = g.run(c.n_eq, c.n_meas)
    pred_g = pred_g.cpu().numpy()
    m1 = mask == 1
    zmin, zmax = o.zrange()
    assert g.counters() == o.counters()                               # every accept/reject decision of 1100 sweeps
    assert np.array_equal(pred_g[~m1], values[~m1])
    assert np.max(np.abs(pred_g[m1] - pred_o[m1])) <= 1e-8 * (zmax - zmin)
    assert abs(e_g - e_o) <= 1e-11
    g.close()
    mae_o, rmse_o = inputs.prediction_errors(pred_o, truth, mask)
    assert mae_o < 0.5 * float(np.mean(np.abs(truth[m1] - values[~m1].mean())))     # it predicts (sanity, not parity)
    _float_mode_gates(mpr, inputs, dv, dm, truth, mask, ("SP",), c.mpr_seed, T_o, c.n_eq, c.n_meas, e_o, se_o,
                      mae_o, rmse_o)


def test_config3_actual_size(mpr, oracle_mod, inputs):
    """BASELINE.json configs[2] as stated: L = 2048 lognormal field (spins crowded near phi = 0, T_hat ~ 1e-3: the
    float-precision stress case), 33 % masked, 1000 + 100 sweeps, all four modes at the oracle's T_hat.
    DP equals the oracle over the whole run; SP, SP_PRECISE and SP_INTRINSIC meet the statistical gates."""
    import torch
    c, values, mask, truth = inputs.make_config(3)
    dv, dm = torch.from_numpy(values).cuda(), torch.from_numpy(mask).cuda()
    o = oracle_mod.Oracle(values=values, mask=mask, seed=c.mpr_seed, threads=oracle_mod.threads_available())
    T_o, _, _ = o.estimate_temperature()
    assert 1e-4 < T_o < 1e-2
    pred_o, e_o, se_o = o.run(c.n_eq, c.n_meas)
    g = mpr.Mpr(dv, dm, seed=c.mpr_seed)
    g.set_temperature(T_o)
    pred_g, e_g, se_g = g.run(c.n_eq, c.n_meas)
    pred_g = pred_g.cpu().numpy()
    m1 = mask == 1
    zmin, zmax = o.zrange()
    assert g.counters() == o.counters()
    assert np.max(np.abs(pred_g[m1] - pred_o[m1])) <= 1e-8 * (zmax - zmin)
    assert abs(e_g - e_o) <= 1e-11
    g.close()
    mae_o, rmse_o = inputs.prediction_errors(pred_o, truth, mask)
    _float_mode_gates(mpr, inputs, dv, dm, truth, mask, ("SP", "SP_PRECISE", "SP_INTRINSIC"), c.mpr_seed, T_o,
                      c.n_eq, c.n_meas, e_o, se_o, mae_o, rmse_o)


@pytest.mark.parametrize("config", [4, 5])
def test_configs_4_and_5_actual_size(mpr, inputs, config):
    """BASELINE.json configs[3] (L = 8192, 66 % masked, SP and SP_INTRINSIC) and configs[4] (L = 16384, 90 %
    masked, all four modes) as stated: T inferred, 2000 + 200 sweeps, prediction error against the held-out
    truth.  The oracle cannot finish these sizes in seconds, so the reference is the GPU DP chain at the same
    T_hat (decision-identical to the oracle wherever the oracle can run: configs 1-3, L = 4100): each float
    mode's e within 3 standard errors of it, MAE and RMSE within 1 % of its."""
    import torch
    c, values, mask, truth = inputs.make_config(config)
    dv, dm, dt = torch.from_numpy(values).cuda(), torch.from_numpy(mask).cuda(), torch.from_numpy(truth).cuda()
    free = dm.bool()
    del values, truth

    def errors(pred):
        d = (pred - dt)[free]
        return float(d.abs().mean()), float(d.pow(2).mean().sqrt())

    g = mpr.Mpr(dv, dm, mode="DP", seed=c.mpr_seed)
    T_hat, e_s, n_trials = g.estimate_temperature()
    assert 1e-4 < T_hat < 1e-1 and 2 <= n_trials <= 22
    pred, e_ref, se_ref = g.run(c.n_eq, c.n_meas)
    mae_ref, rmse_ref = errors(pred)
    assert torch.equal(pred[~free], dv[~free])                         # measured values come back bit-exact
    g.close()
    del g, pred
    base = float((dt[free] - dv[~free].mean()).abs().mean())
    assert mae_ref < 0.5 * base                                        # it predicts (sanity, not parity)
    for mode in c.modes:
        if mode == "DP":
            continue
        g = mpr.Mpr(dv, dm, mode=mode, seed=c.mpr_seed)
        g.set_temperature(T_hat)
        pred, e, se = g.run(c.n_eq, c.n_meas)
        mae, rmse = errors(pred)
        g.close()
        del g, pred
        assert abs(e - e_ref) <= 3.0 * math.hypot(se, se_ref), (mode, e, e_ref, se, se_ref)
        assert abs(mae / mae_ref - 1.0) <= 0.01, (mode, mae, mae_ref)
        assert abs(rmse / rmse_ref - 1.0) <= 0.01, (mode, rmse, rmse_ref)


# --------------------------------------------------------------------------- large grids
def test_dp_large_ragged_grid_matches_oracle(mpr, oracle_mod, inputs):
    """L = 4100 (69 x 103 DP tiles, ragged tail in both directions, plane padding columns): every
    site after the tiled quench passes and 2 hybrid sweeps, and the accepted-move count."""
    L = 4100
    values, mask, _ = make(inputs, L, 64.0, 21, 0.9)
    g = mpr.Mpr(values, mask, seed=1234)
    o = oracle_mod.Oracle(values=values, mask=mask, seed=1234, threads=oracle_mod.threads_available())
    g.set_quench(2)
    o.set_quench(2)
    g.set_temperature(0.004)
    o.set_temperature(0.004)
    g.sweep(2)
    o.hybrid_sweeps(2)
    sg, so = g.get_state().cpu().numpy(), o.get_state()
    assert phi_diff(sg, so) <= PHI_TOL
    assert g.counters() == o.counters()
    assert abs(g.energy()[1] - o.energy()[1]) <= 1e-10


@pytest.fixture(scope="module")
def config5(inputs):
    """BASELINE.json configs[4] on the device, generated once for all full-size cases (15 s, 2 GiB)."""
    import torch
    c, values, mask, truth = inputs.make_config(5)
    return c, torch.from_numpy(values).cuda(), torch.from_numpy(mask).cuda(), int(mask.sum())


@pytest.mark.parametrize("mode", ["SP_INTRINSIC", "SP_PRECISE", "SP", "DP"])
def test_bench_configuration_full_size_properties(mpr, config5, mode):
    """BASELINE.json configs[4] (L = 16384, 90 % masked) in the launch configurations bench.py times
    (every precision mode, tiled, one hybrid sweep per launch).  The oracle cannot finish this size in
    seconds, so the full grid is checked through what holds at any size: the tiled kernel equals the
    plain per-pass kernels bit for bit (spins, accepted moves), measured spins never move, every
    angle stays in [0, 2 pi], the fused energy sample equals the plain energy kernel's, and the
    prediction leaves measured sites bit-exact."""
    import torch
    c, d_values, d_mask, n_free = config5
    out = {}
    for path in ("TILED", "PLAIN", "STRIP"):
        g = mpr.Mpr(d_values, d_mask, mode=mode, seed=c.mpr_seed)
        g.set_path(path)
        g.set_quench(2)
        g.set_temperature(1.1e-3)
        s0 = g.get_state()
        g.sweep(3)
        s1 = g.get_state()
        cnt = g.counters()
        pred, e, se = g.run(0, 2)
        out[path] = (s1, cnt, g.series(), pred)
        if path == "STRIP":                                           # bench.py's path
            m0 = d_mask == 0
            assert torch.equal(s0[m0], s1[m0])                       # measured spins never move
            assert float(s1.min()) >= 0.0 and float(s1.max()) <= TWO_PI + 1e-15
            assert torch.equal(pred[m0], d_values[m0])               # measured values come back bit-exact
            free = pred[~m0]
            assert bool(torch.isfinite(free).all())
            zmin, zmax = g.info()["z_min"], g.info()["z_max"]
            assert float(free.min()) >= zmin - 1e-9 and float(free.max()) <= zmax + 1e-9   # R1 confines predictions
            assert cnt[1] == 3 * n_free and cnt[0] > 0
        g.close()
        del g
    for path in ("TILED", "STRIP"):
        assert torch.equal(out[path][0], out["PLAIN"][0]), path
        assert out[path][1] == out["PLAIN"][1], path
        np.testing.assert_allclose(out[path][2], out["PLAIN"][2], rtol=0, atol=1e-12)
        assert torch.equal(out[path][3], out["PLAIN"][3]), path
    if mode == "SP_INTRINSIC":
        # bench.py also times the step with two sweeps per launch (`two_sweeps_per_launch`): 5 sweeps at depth 2 =
        # launches of 2 + 2 + 1 sweeps, against the per-pass kernels
        res = {}
        for path, k in (("STRIP", 2), ("PLAIN", 1)):
            g = mpr.Mpr(d_values, d_mask, mode=mode, seed=c.mpr_seed)
            g.set_path(path); g.set_fused_sweeps(k); g.set_quench(2); g.set_temperature(1.1e-3)
            g.sweep(5)
            res[path] = (g.get_state(), g.counters())
            g.close()
        assert torch.equal(res["STRIP"][0], res["PLAIN"][0]) and res["STRIP"][1] == res["PLAIN"][1]
