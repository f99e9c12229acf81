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
