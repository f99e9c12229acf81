"""Rectangular grids (include/mpr.h: mpr_create_rect): the CUDA path on Lx x Ly grids against the oracle
(DP: identical decisions, |dphi| <= 1e-9) and, in the float modes, every kernel path against the per-pass PLAIN path
(bit-identical).  Shapes: wide, tall, odd sides, a single row, a single column, strips with a ragged tail."""
import math

import numpy as np
import pytest

pytestmark = pytest.mark.gpu

PHI_TOL = 1e-9
SHAPES = [(37, 150), (150, 37), (1, 64), (64, 1), (130, 257), (3, 2), (20, 515)]      # (Ly rows, Lx columns)


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


@pytest.mark.parametrize("shape", SHAPES, ids=["%dx%d" % s for s in SHAPES])
def test_rect_setup_and_energies_match_oracle(mpr, oracle_mod, inputs, shape):
    Ly, Lx = shape
    values, mask, _ = inputs.make_rect_problem(Ly, Lx, 6.0, 21, 0.6)
    g = mpr.Mpr(values, mask, seed=7)
    o = oracle_mod.Oracle(values=values, mask=mask, seed=7)
    info = g.info()
    assert (info["z_min"], info["z_max"]) == o.zrange() and info["n_free"] == int(mask.sum())
    try:
        es_o, n_o = o.sample_energy()
    except oracle_mod.OracleError:
        es_o = None
    if es_o is not None:
        es_g, n_g = g.sample_energy()
        assert n_g == n_o and abs(es_g - es_o) <= 1e-12 * abs(es_o)
    assert phi_diff(g.get_state().cpu().numpy(), o.get_state()) <= 1e-12          # R8: uniform start + quench passes
    H_g, e_g = g.energy()
    H_o, e_o = o.energy()
    assert abs(H_g - H_o) <= 1e-11 * max(1.0, abs(H_o)) and abs(e_g - e_o) <= 1e-11


@pytest.mark.parametrize("schedule", ["R4", "SITE_FUSED"])
@pytest.mark.parametrize("path", ["PLAIN", "LIST", "TILED", "STRIP"])
@pytest.mark.parametrize("shape", SHAPES, ids=["%dx%d" % s for s in SHAPES])
def test_rect_dp_sweeps_match_oracle(mpr, oracle_mod, inputs, shape, path, schedule):
    if schedule == "SITE_FUSED" and path == "TILED":
        pytest.skip("the tiled kernels carry the R4 order only")
    Ly, Lx = shape
    values, mask, _ = inputs.make_rect_problem(Ly, Lx, 6.0, 22, 0.75)
    g = mpr.Mpr(values, mask, seed=313)
    o = oracle_mod.Oracle(values=values, mask=mask, seed=313)
    for h in (g, o):
        h.set_temperature(0.05)
        h.set_schedule(schedule)
    g.set_path(path)
    g.sweep(6)
    o.hybrid_sweeps(6)
    sg, so = g.get_state().cpu().numpy(), o.get_state()
    assert sg.shape == (Ly, Lx)
    assert phi_diff(sg, so) <= PHI_TOL
    assert g.counters() == o.counters()
    assert sg.min() >= 0.0 and sg.max() <= 2.0 * math.pi + 1e-15


@pytest.mark.parametrize("shape", [(37, 150), (150, 37), (130, 257), (1, 64), (64, 1)], ids=lambda s: "%dx%d" % s)
def test_rect_dp_run_matches_oracle(mpr, oracle_mod, inputs, shape):
    """mpr_run on a rectangular grid: energy series, prediction (mean of phi mapped back), temperature matching."""
    Ly, Lx = shape
    values, mask, _ = inputs.make_rect_problem(Ly, Lx, 6.0, 23, 0.5)
    g = mpr.Mpr(values, mask, seed=99)
    o = oracle_mod.Oracle(values=values, mask=mask, seed=99)
    if min(Ly, Lx) > 1:
        T_g, T_o = g.estimate_temperature()[0], o.estimate_temperature()[0]
        assert abs(T_g - T_o) <= 1e-9 * T_o
    else:
        g.set_temperature(0.03); o.set_temperature(0.03)
    for path in ("STRIP", "TILED", "PLAIN"):
        g.set_path(path)
        g.reset_chain(0); o.reset_chain(0)
        pred_g, e_g, se_g = g.run(12, 9)
        pred_o, e_o, se_o = o.run(12, 9)
        assert abs(e_g - e_o) <= 1e-11 and abs(se_g - se_o) <= 1e-11, path
        pg = pred_g.cpu().numpy()
        assert pg.shape == (Ly, Lx)
        zr = o.zrange()
        assert np.max(np.abs(pg - pred_o)) <= 1e-9 * (zr[1] - zr[0]), path
        m0 = mask == 0
        assert np.array_equal(pg[m0], values[m0])


@pytest.mark.parametrize("mode", ["SP_INTRINSIC", "SP_PRECISE", "SP", "HP", "DS_INTRINSIC"])
@pytest.mark.parametrize("shape", [(37, 150), (150, 37), (130, 257), (1, 64), (64, 1), (20, 515)], ids=lambda s: "%dx%d" % s)
def test_rect_float_paths_are_bit_identical(mpr, inputs, shape, mode):
    import torch
    Ly, Lx = shape
    values, mask, _ = inputs.make_rect_problem(Ly, Lx, 6.0, 24, 0.8)
    ref = {}
    for path, k, sched in [("PLAIN", 1, "R4"), ("TILED", 1, "R4"), ("STRIP", 1, "R4"), ("STRIP", 2, "R4"), ("LIST", 1, "R4"),
                           ("PLAIN", 1, "SITE_FUSED"), ("STRIP", 1, "SITE_FUSED"), ("STRIP", 2, "SITE_FUSED"),
                           ("LIST", 1, "SITE_FUSED")]:
        g = mpr.Mpr(values, mask, mode=mode, seed=5)
        g.set_path(path); g.set_fused_sweeps(k); g.set_schedule(sched)
        g.set_temperature(0.02)
        g.sweep(4)
        st, cnt = g.get_state(), g.counters()
        pred, e, se = g.run(3, 4)
        if path == "PLAIN":
            ref[sched] = (st, cnt, pred, e)
        else:
            r = ref[sched]
            assert torch.equal(st, r[0]) and cnt == r[1], (path, k, sched)
            assert torch.equal(torch.nan_to_num(pred), torch.nan_to_num(r[2])), (path, k, sched)
            assert abs(e - r[3]) <= 2e-6 * abs(r[3]), (path, k, sched)
        g.close()


def test_rect_host_call_and_argument_checks(mpr, oracle_mod, inputs):
    Ly, Lx = 45, 120
    values, mask, _ = inputs.make_rect_problem(Ly, Lx, 6.0, 25, 0.5)
    pred, e, se, T, nl = mpr.predict_host(values, mask, mode="DP", seed=3, T=0.05, n_eq=8, n_meas=6)
    o = oracle_mod.Oracle(values=values, mask=mask, seed=3)
    o.set_temperature(0.05)
    pred_o, e_o, se_o = o.run(8, 6)
    zr = o.zrange()
    assert pred.shape == (Ly, Lx) and abs(e - e_o) <= 1e-11 and np.max(np.abs(pred - pred_o)) <= 1e-9 * (zr[1] - zr[0])
    import ctypes as C
    n = C.c_size_t()
    lib = mpr.lib()
    assert lib.mpr_workspace_bytes_rect(0, 5, C.byref(n)) == mpr.ERR_INVALID_ARG
    assert lib.mpr_workspace_bytes_rect(1, 1, C.byref(n)) == mpr.ERR_INVALID_ARG
    assert lib.mpr_workspace_bytes_rect(40000, 2, C.byref(n)) == mpr.ERR_INVALID_ARG
    assert lib.mpr_workspace_bytes_rect(1, 2, C.byref(n)) == mpr.MPR_OK and n.value > 0
    assert mpr.workspace_bytes((7, 7)) == mpr.workspace_bytes(7)
