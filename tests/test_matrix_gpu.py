"""The paper's eight precision settings (X_S X_E X_F): spin storage, energy variable, functions, each D or S.
X_S, X_F select the kernel mode, X_E the arithmetic of the energy reduction (include/mpr.h, mpr_set_precision_triple)."""
import math

import numpy as np
import pytest

pytestmark = pytest.mark.gpu


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


@pytest.mark.parametrize("triple", ["DDD", "DSD", "DDS", "SDD", "SDS", "DSS", "SSD", "SSS"])
def test_every_setting_is_path_independent(mpr, inputs, triple):
    """Spins, counters, prediction bit-identical on the PLAIN, TILED and STRIP paths; energies to the rounding of the
    chosen energy variable."""
    values, mask, _ = inputs.make_problem(300, 12.0, 4, 0.9, False)
    out = []
    for path in ("PLAIN", "TILED", "STRIP"):
        g = mpr.Mpr(values, mask, seed=5)
        g.set_precision_triple(triple)
        g.set_path(path)
        g.set_temperature(0.05)
        g.sweep(6)
        pred, e, se = g.run(2, 4)
        out.append((g.get_state().cpu().numpy(), g.counters(), pred.cpu().numpy(), g.series()))
        g.close()
    for o in out[1:]:
        assert np.array_equal(o[0], out[0][0]) and o[1] == out[0][1]
        assert np.array_equal(o[2], out[0][2])
        tol = 3e-6 if triple[1] == "S" else 1e-12          # a float energy variable: the summation order shows
        np.testing.assert_allclose(o[3], out[0][3], rtol=0, atol=tol)
    if triple[1] == "S":
        s = out[1][3]
        assert np.array_equal(s, s.astype(np.float32).astype(np.float64))      # the reported e_n IS a float


@pytest.mark.parametrize("xs_xf", ["DD", "SD", "DS", "SS"])
def test_energy_variable_precision(mpr, inputs, xs_xf):
    """X_E only changes how the energy of a state is evaluated: the same state, X_E = D against X_E = S."""
    values, mask, _ = inputs.make_problem(512, 16.0, 6, 0.9, False)
    g = mpr.Mpr(values, mask, seed=3)
    g.set_precision_triple(xs_xf[0] + "D" + xs_xf[1])
    g.set_temperature(0.02)
    g.sweep(20)
    st = g.get_state().cpu().numpy()
    e_d = g.energy()[1]
    g.set_energy_precision(1)
    assert np.array_equal(g.get_state().cpu().numpy(), st)       # the chain is untouched
    e_s = g.energy()[1]
    assert e_s == float(np.float32(e_s))
    assert 0.0 < abs(e_s - e_d) < 2e-6 * abs(e_d)                 # float rounding of ~5e5 bond terms, and it is visible
    g.set_energy_precision(0)
    assert g.energy()[1] == e_d


def test_double_storage_float_functions_statistics(mpr, oracle_mod, inputs):
    """MPR_DS_INTRINSIC (the paper's D.S settings): float arithmetic on double-stored spins, judged like the other float
    modes -- e within 3 standard errors of the DP oracle's, MAE / RMSE within 1 %."""
    L, T = 256, 0.03
    values, mask, truth = inputs.make_problem(L, 16.0, 1, 0.66, False)
    o = oracle_mod.Oracle(values=values, mask=mask, seed=1001, threads=oracle_mod.threads_available())
    o.set_temperature(T)
    pred_o, e_o, se_o = o.run(300, 200)
    mae_o, rmse_o = inputs.prediction_errors(pred_o, truth, mask)
    es, errs = [], []
    for seed in range(1, 9):
        g = mpr.Mpr(values, mask, mode="DS_INTRINSIC", seed=seed)
        g.set_temperature(T)
        pred, e, se = g.run(300, 200)
        es.append(e)
        errs.append(inputs.prediction_errors(pred.cpu().numpy(), truth, mask))
        g.close()
    e_se = float(np.std(es, ddof=1) / math.sqrt(len(es)))
    assert abs(float(np.mean(es)) - e_o) <= 3.0 * math.hypot(e_se, se_o) + 1e-6
    assert abs(float(np.mean([m for m, _ in errs])) / mae_o - 1.0) <= 0.01
    assert abs(float(np.mean([r for _, r in errs])) / rmse_o - 1.0) <= 0.01


def test_triple_argument_validation(mpr, inputs):
    values, mask, _ = inputs.make_problem(32, 4.0, 1, 0.5, False)
    g = mpr.Mpr(values, mask)
    for bad in ("DD", "DDDD", "XDD", "ddd"):
        with pytest.raises(mpr.MprError) as ei:
            g.set_precision_triple(bad)
        assert ei.value.code == mpr.ERR_INVALID_ARG


# --------------------------------------------------------------------------- compacted site lists, structured gaps
@pytest.mark.parametrize("mode", ["DP", "SP_INTRINSIC"])
@pytest.mark.parametrize("schedule", ["R4", "SITE_FUSED"])
def test_list_path_equals_plain(mpr, inputs, mode, schedule):
    """north_star (a): the compacted per-colour lists of prediction sites.  The LIST path visits exactly the sites
    the PLAIN path finds by testing mask bits, with the same moves: spins, counters, prediction bit-identical --
    at a small and at a large masked fraction, on a ragged grid."""
    for L, f in ((131, 0.33), (300, 0.9)):
        values, mask, _ = inputs.make_problem(L, 12.0, 4, f, False)
        out = []
        for path in ("PLAIN", "LIST"):
            g = mpr.Mpr(values, mask, mode=mode, seed=5)
            g.set_path(path)
            g.set_schedule(schedule)
            g.set_temperature(0.05)
            g.sweep(7)
            pred, e, se = g.run(2, 3)
            out.append((g.get_state().cpu().numpy(), g.counters(), pred.cpu().numpy(), g.series()))
            g.close()
        assert np.array_equal(out[0][0], out[1][0]) and out[0][1] == out[1][1]
        assert np.array_equal(out[0][2], out[1][2]) and np.array_equal(out[0][3], out[1][3])


@pytest.mark.parametrize("kind", ["clouds", "tracks"])
def test_structured_gaps_match_oracle(mpr, oracle_mod, inputs, kind):
    """Clustered gaps: whole warps and tiles without a prediction site next to fully masked ones.
    DP on every path against the oracle: identical decisions, |dphi| <= 1e-9; the float mode path-independent."""
    L = 260
    values, mask, truth = inputs.make_structured_problem(L, 16.0, 3, 0.6, kind)
    assert 0.4 < mask.mean() < 0.8
    o = oracle_mod.Oracle(values=values, mask=mask, seed=21)
    o.set_temperature(0.04)
    o.hybrid_sweeps(8)
    so, cnt_o = o.get_state(), o.counters()
    for path in ("PLAIN", "LIST", "TILED", "STRIP"):
        g = mpr.Mpr(values, mask, mode="DP", seed=21)
        g.set_path(path)
        g.set_temperature(0.04)
        g.sweep(8)
        assert float(np.max(np.abs(g.get_state().cpu().numpy() - so))) <= 1e-9, path
        assert g.counters() == cnt_o, path
        g.close()
    ref = None
    for path in ("PLAIN", "LIST", "TILED", "STRIP"):
        g = mpr.Mpr(values, mask, mode="SP_INTRINSIC", seed=21)
        g.set_path(path)
        g.set_temperature(0.04)
        pred, e, se = g.run(30, 20)
        cur = (g.get_state().cpu().numpy(), g.counters(), pred.cpu().numpy())
        g.close()
        if ref is None:
            ref = cur
            mae, _ = inputs.prediction_errors(cur[2], truth, mask)
            base = float(np.mean(np.abs(truth[mask == 1] - np.nanmean(values))))
            assert mae < base                               # it predicts into the gaps (sanity)
        else:
            assert np.array_equal(cur[0], ref[0]) and cur[1] == ref[1] and np.array_equal(cur[2], ref[2]), path


# --------------------------------------------------------------------------- half-precision storage
def test_half_precision_storage(mpr, inputs):
    """MPR_HP: spins stored as two fp16 (4 bytes per spin), float arithmetic.  Judged like the float modes on the
    prediction (MAE / RMSE within 1 % of DP); the stored vectors carry a 5e-4 relative rounding, so the energy
    is only held to 0.2 % of its thermal part, |e - e_DP| <= 3e-5 at T = 0.03 (measured with 16 seeds: +1.3e-6 +- 3e-6
    there, +1.4e-7 +- 3e-8 at T = 1.1e-3, i.e. a visible bias at low T)."""
    L, T = 512, 0.03
    values, mask, truth = inputs.make_problem(L, 32.0, 1, 0.66, False)
    res = {}
    for mode in ("DP", "HP"):
        es, errs = [], []
        for seed in (1, 2, 3, 4, 5, 6):
            g = mpr.Mpr(values, mask, mode=mode, seed=seed)
            g.set_temperature(T)
            s0 = g.get_state().cpu().numpy()
            pred, e, se = g.run(300, 150)
            s1 = g.get_state().cpu().numpy()
            m0 = mask == 0
            assert np.array_equal(s0[m0], s1[m0])                      # measured spins never move
            assert s1.min() >= 0.0 and s1.max() <= 2.0 * math.pi + 1e-12
            assert np.array_equal(pred.cpu().numpy()[m0], values[m0])
            es.append(e)
            errs.append(inputs.prediction_errors(pred.cpu().numpy(), truth, mask))
            g.close()
        res[mode] = (float(np.mean(es)), float(np.mean([a for a, _ in errs])), float(np.mean([b for _, b in errs])))
    assert abs(res["HP"][0] - res["DP"][0]) <= 3e-5
    # the fused STRIP kernels (two halo lanes per side, so that every TMA box row starts on a 16-byte boundary at 4 bytes
    # per plane column) give the same chain as the per-pass kernels; TILED asks are served by STRIP
    ref = None
    for path in ("PLAIN", "LIST", "STRIP", "TILED"):
        g = mpr.Mpr(values, mask, mode="HP", seed=3)
        g.set_path(path)
        g.set_temperature(T)
        g.sweep(5)
        pred, e, se = g.run(2, 3)
        cur = (g.get_state().cpu().numpy(), g.counters(), pred.cpu().numpy())
        g.close()
        if ref is None:
            ref = cur
        else:
            assert np.array_equal(cur[0], ref[0]) and cur[1] == ref[1] and np.array_equal(cur[2], ref[2]), path
    assert abs(res["HP"][1] / res["DP"][1] - 1.0) <= 0.01
    assert abs(res["HP"][2] / res["DP"][2] - 1.0) <= 0.01


# --------------------------------------------------------------------------- site-fused schedule (R4b) vs the oracle
@pytest.mark.parametrize("L,f,T", [(97, 0.9, 0.02), (250, 0.66, 0.3)])
def test_site_fused_schedule_matches_oracle(mpr, oracle_mod, inputs, L, f, T):
    """DP, pass order MET c0, OR c0, MET c1, OR c1 (the oracle's `SITE_FUSED` flag, pinned by the single-site and
    two-site tests of tests/test_oracle_pins.py): identical decisions and |dphi| <= 1e-9 after 10 sweeps on the
    PLAIN, LIST and STRIP paths (one and two sweeps per launch), then a measured run."""
    values, mask, _ = inputs.make_problem(L, 8.0, 3, f, False)
    o = oracle_mod.Oracle(values=values, mask=mask, seed=1000)
    o.set_schedule("SITE_FUSED")
    o.set_temperature(T)
    o.hybrid_sweeps(10)
    so, cnt_o = o.get_state(), o.counters()
    pred_o, e_o, _ = o.run(3, 5)
    for path, k in (("PLAIN", 1), ("LIST", 1), ("STRIP", 1), ("STRIP", 2)):
        g = mpr.Mpr(values, mask, mode="DP", seed=1000)
        g.set_path(path)
        g.set_schedule("SITE_FUSED")
        g.set_fused_sweeps(k)
        g.set_temperature(T)
        g.sweep(10)
        assert float(np.max(np.abs(g.get_state().cpu().numpy() - so))) <= 1e-9, (path, k)
        assert g.counters() == cnt_o, (path, k)
        pred, e, _ = g.run(3, 5)
        m1 = mask == 1
        assert float(np.max(np.abs(pred.cpu().numpy()[m1] - pred_o[m1]))) <= 1e-8 * 100.0
        assert abs(e - e_o) <= 1e-11
        g.close()
    # and it IS a different chain from R4 (same random numbers, other order)
    g = mpr.Mpr(values, mask, mode="DP", seed=1000)
    g.set_temperature(T)
    g.sweep(10)
    assert float(np.max(np.abs(g.get_state().cpu().numpy() - so))) > 1e-3


# --------------------------------------------------------------------------- general q
@pytest.mark.parametrize("q", [0.3, 0.1])
@pytest.mark.parametrize("schedule", ["R4", "SITE_FUSED"])
def test_general_q_matches_oracle(mpr, oracle_mod, inputs, q, schedule):
    """q < 1/2: set-up (sample energy), R8 initialisation (the quench clips at phi = 2 pi), 10 hybrid sweeps and a
    measured run in DP against the oracle with the same q -- identical decisions, |dphi| <= 1e-9 -- on the PLAIN and
    LIST paths; asking for a fused path still works (the context routes itself to the per-pass kernels)."""
    values, mask, _ = inputs.make_problem(120, 8.0, 3, 0.8, False)
    o = oracle_mod.Oracle(values=values, mask=mask, seed=1000)
    o.set_q(q)
    o.set_schedule(schedule)
    o.set_temperature(0.05)
    es_o, n_o = o.sample_energy()
    s_init = o.get_state()
    o.hybrid_sweeps(10)
    so, cnt_o = o.get_state(), o.counters()
    pred_o, e_o, _ = o.run(3, 5)
    for path in ("PLAIN", "LIST", "STRIP"):
        g = mpr.Mpr(values, mask, mode="DP", seed=1000)
        g.set_q(q)
        g.set_path(path)
        g.set_schedule(schedule)
        g.set_temperature(0.05)
        es_g, n_g = g.sample_energy()
        assert n_g == n_o and abs(es_g - es_o) <= 1e-12
        assert float(np.max(np.abs(g.get_state().cpu().numpy() - s_init))) <= 1e-9
        g.sweep(10)
        sg = g.get_state().cpu().numpy()
        assert float(np.max(np.abs(sg - so))) <= 1e-9, path
        assert sg.min() >= 0.0 and sg.max() <= 2.0 * math.pi + 1e-12
        assert g.counters() == cnt_o, path
        pred, e, _ = g.run(3, 5)
        m1 = mask == 1
        assert float(np.max(np.abs(pred.cpu().numpy()[m1] - pred_o[m1]))) <= 1e-6
        assert abs(e - e_o) <= 1e-11
        g.close()
    with pytest.raises(mpr.MprError):
        mpr.Mpr(values, mask).set_q(0.6)


@pytest.mark.parametrize("mode", ["SP_INTRINSIC", "SP_PRECISE"])
def test_general_q_float_modes_sample_the_exact_density(mpr, mode):
    """Isolated free sites with identical measured neighbourhoods at q = 0.25: chi^2 of the pooled samples against
    p(phi) ~ exp(sum_j cos[q (phi - phi_j)] / T) (the density piles up against phi = 2 pi for these neighbours, so the
    upper range test is exercised)."""
    q, T, L = 0.25, 0.3, 302
    nb = {(-1, 0): 5.3, (1, 0): 6.0, (0, -1): 4.4, (0, 1): 5.8}
    rng = np.random.default_rng(3)
    z = rng.uniform(0.5, 5.5, (L, L))
    mask = np.zeros((L, L), dtype=np.uint8)
    sites = [(x, y) for y in range(2, L - 2, 3) for x in range(1, L - 3, 3)]
    for (x, y) in sites:
        mask[y, x] = 1
        for (dx, dy), a in nb.items():
            z[y + dy, x + dx] = a
    z[L // 2, L - 1], z[L // 2 + 2, L - 1] = 0.0, 2.0 * math.pi          # anchors of the R1 map: phi = z
    g = mpr.Mpr(z, mask, mode=mode, seed=9)
    g.set_q(q)
    g.set_temperature(T)
    g.sweep(60)
    ys, xs = np.array([s[1] for s in sites]), np.array([s[0] for s in sites])
    snaps = []
    for _ in range(50):
        g.sweep(6)
        snaps.append(g.get_state().cpu().numpy()[ys, xs])
    samples = np.concatenate(snaps)
    grid = np.linspace(0.0, 2.0 * math.pi, 400001)
    logw = sum(np.cos(q * (grid - a)) for a in nb.values()) / T
    w = np.exp(logw - logw.max())
    cdf = np.concatenate([[0.0], np.cumsum(0.5 * (w[1:] + w[:-1]) * np.diff(grid))])
    cdf /= cdf[-1]
    nbins = 40
    edges = np.concatenate([[0.0], np.interp(np.arange(1, nbins) / nbins, cdf, grid), [2.0 * math.pi + 1e-9]])
    cnt, _ = np.histogram(samples, bins=edges)
    assert cnt.sum() == samples.size
    chi2 = float(((cnt - samples.size / nbins) ** 2 / (samples.size / nbins)).sum())
    assert chi2 < 85.0, chi2
    assert float(np.mean(samples > 6.0)) > 0.05            # the mass near the upper end of the range is really there
