"""Slab decomposition (paper_1910_08448_b200/slabs.py, include/mpr.h "Slabs") on ONE GPU: G slab contexts
worked off in turn with halo refreshes must reproduce the single-context run on the whole grid bit for bit (spins,
accepted moves, prediction) and its energies up to the order of the final sums; in DP they match the oracle like the
single context does."""
import numpy as np
import pytest

pytestmark = pytest.mark.gpu

PHI_TOL = 1e-9


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


@pytest.fixture(scope="module")
def slabs():
    from paper_1910_08448_b200 import slabs as s
    return s


def whole(mpr, values, mask, mode, seed, path, schedule, T, n_eq, n_meas):
    g = mpr.Mpr(values, mask, mode=mode, seed=seed)
    g.set_path(path); g.set_schedule(schedule); g.set_temperature(T)
    pred, e, se = g.run(n_eq, n_meas)
    out = (g.get_state().cpu().numpy(), g.counters()[0], g.series(), pred.cpu().numpy(), e, se, g.sample_energy(), g.info())
    g.close()
    return out


@pytest.mark.parametrize("mode,path,schedule", [("DP", "PLAIN", "R4"), ("DP", "TILED", "R4"), ("DP", "STRIP", "SITE_FUSED"),
                                                ("SP_INTRINSIC", "STRIP", "R4"), ("SP_INTRINSIC", "TILED", "R4"),
                                                ("SP_INTRINSIC", "LIST", "SITE_FUSED"), ("SP", "STRIP", "R4"),
                                                ("HP", "STRIP", "R4")])
@pytest.mark.parametrize("count,halo", [(1, 8), (2, 4), (3, 8), (5, 12)])
def test_slabs_reproduce_the_single_context(mpr, inputs, slabs, mode, path, schedule, count, halo):
    Ly, Lx = 190, 141
    values, mask, _ = inputs.make_rect_problem(Ly, Lx, 7.0, 51, 0.7)
    T, n_eq, n_meas = 0.04, 7, 6
    st_w, acc_w, series_w, pred_w, e_w, se_w, (es_w, np_w), info_w = whole(mpr, values, mask, mode, 77, path, schedule, T, n_eq, n_meas)
    ss = slabs.make_slab_set(values, mask, count, halo=halo, mode=mode, seed=77, path=path, schedule=schedule)
    assert (ss.z_min, ss.z_max) == (info_w["z_min"], info_w["z_max"]) and ss.n_free == info_w["n_free"]
    assert ss.n_pairs == np_w and abs(ss.e_sample - es_w) <= 1e-12 * abs(es_w)
    ss.set_temperature(T)
    ss.reset_chain(0)
    series, e, se = ss.run(n_eq, n_meas)
    assert np.array_equal(ss.state(), st_w)                      # every spin, bit for bit
    assert ss.accepted() == acc_w
    tol = 1e-12 if mode != "HP" else 1e-12
    assert np.max(np.abs(series - np.asarray(series_w))) <= tol * 2.0, (series, series_w)
    assert abs(e - e_w) <= 2e-12 and abs(se - se_w) <= 2e-12
    pw, ps = np.nan_to_num(pred_w, nan=-1.0), np.nan_to_num(ss.prediction(), nan=-1.0)
    assert np.array_equal(ps, pw)


def test_slabs_dp_match_the_oracle(mpr, oracle_mod, inputs, slabs):
    Ly, Lx = 120, 97
    values, mask, _ = inputs.make_rect_problem(Ly, Lx, 6.0, 52, 0.8)
    o = oracle_mod.Oracle(values=values, mask=mask, seed=5)
    o.set_temperature(0.06)
    ss = slabs.make_slab_set(values, mask, 3, halo=8, mode="DP", seed=5, path="STRIP")
    ss.set_temperature(0.06)
    ss.reset_chain(0)
    pred_o, e_o, se_o = o.run(9, 8)
    series, e, se = ss.run(9, 8)
    assert np.max(np.abs(ss.state() - o.get_state())) <= PHI_TOL
    assert ss.accepted() == o.counters()[0]
    assert abs(e - e_o) <= 1e-11 and abs(se - se_o) <= 1e-11
    zr = o.zrange()
    assert np.max(np.abs(ss.prediction() - pred_o)) <= 1e-9 * (zr[1] - zr[0])


def test_slabs_temperature_matching(mpr, inputs, slabs):
    """R6 over slabs: every trial chain runs on all slabs, the energies are the summed parts."""
    Ly, Lx = 96, 96
    values, mask, _ = inputs.make_rect_problem(Ly, Lx, 8.0, 53, 0.66)
    g = mpr.Mpr(values, mask, mode="DP", seed=9)
    T_w = g.estimate_temperature()[0]
    g.close()
    ss = slabs.make_slab_set(values, mask, 2, halo=8, mode="DP", seed=9)
    T_s = ss.estimate_temperature()
    assert abs(T_s - T_w) <= 1e-9 * T_w
    assert ss.exchanges > 0


def test_slab_argument_checks(mpr, inputs, slabs):
    values, mask, _ = inputs.make_rect_problem(40, 33, 5.0, 54, 0.5)
    g = mpr.Mpr(values, mask)
    for args in [(1, 0, 40, 0.0, 1.0, 100.0), (0, 5, 5, 0.0, 1.0, 100.0), (0, 0, 41, 0.0, 1.0, 100.0), (0, 0, 40, 1.0, 1.0, 100.0),
                 (-2, 0, 40, 0.0, 1.0, 100.0)]:
        with pytest.raises(mpr.MprError) as ei:
            g.set_slab(*args)
        assert ei.value.code == mpr.ERR_INVALID_ARG
    with pytest.raises(ValueError):
        slabs.plan_slabs(40, 4, 12)
    with pytest.raises(ValueError):
        slabs.plan_slabs(40, 2, 6)
    plans = slabs.plan_slabs(101, 4, 8)
    assert plans[0].own_begin_g == 0 and plans[-1].own_end_g == 101
    assert all(p.own_begin_g % 2 == 0 and p.row0_g % 2 == 0 for p in plans)
    assert all(a.own_end_g == b.own_begin_g for a, b in zip(plans, plans[1:]))


def test_slabs_at_a_strip_kernel_size(mpr, inputs, slabs):
    """L = 4096 (where MPR_PATH_AUTO picks the strip kernels), 3 slabs of unequal height, the library's 32 quench passes
    by the strip quench kernel with halo refreshes in between."""
    L = 4096
    values, mask, _ = inputs.make_problem(L, 64.0, 55, 0.9)
    g = mpr.Mpr(values, mask, mode="SP_INTRINSIC", seed=8)
    g.set_temperature(0.002)
    pred_w, e_w, se_w = g.run(6, 4)
    st_w, acc_w = g.get_state().cpu().numpy(), g.counters()[0]
    g.close()
    ss = slabs.make_slab_set(values, mask, 3, halo=8, mode="SP_INTRINSIC", seed=8)
    ss.set_temperature(0.002)
    ss.reset_chain(0)
    series, e, se = ss.run(6, 4)
    assert np.array_equal(ss.state(), st_w) and ss.accepted() == acc_w
    assert abs(e - e_w) <= 2e-12
    assert np.array_equal(np.nan_to_num(ss.prediction(), nan=-1.0), np.nan_to_num(pred_w.cpu().numpy(), nan=-1.0))


@pytest.mark.parametrize("mode,schedule", [("SP_INTRINSIC", "R4"), ("SP_INTRINSIC", "SITE_FUSED"), ("DP", "R4"), ("HP", "R4")])
@pytest.mark.parametrize("count", [2, 3, 4])
def test_peer_mode_reproduces_the_single_context(mpr, inputs, slabs, mode, schedule, count):
    """mpr_set_peers: every strip launch writes its 4 edge rows straight into the neighbours' halo rows (peer memory) and
    stores its own rows only -- no export / import launches at all.  Same result as the single context, bit for bit."""
    Ly, Lx = 190, 141
    values, mask, _ = inputs.make_rect_problem(Ly, Lx, 7.0, 56, 0.7)
    T, n_eq, n_meas = 0.04, 7, 6
    st_w, acc_w, series_w, pred_w, e_w, se_w, _, _ = whole(mpr, values, mask, mode, 78, "STRIP", schedule, T, n_eq, n_meas)
    ss = slabs.make_slab_set(values, mask, count, halo=4, mode=mode, seed=78, path="STRIP", schedule=schedule, peer=True)
    ss.set_temperature(T)
    ss.reset_chain(0)
    launches0 = sum(s.ctx.launches() for s in ss.slabs.values())
    series, e, se = ss.run(n_eq, n_meas)
    # one strip launch per slab and sweep, plus the energy reduction of each measuring sweep: nothing else ran
    assert sum(s.ctx.launches() for s in ss.slabs.values()) - launches0 == count * (n_eq + 2 * n_meas)
    assert ss.exchanges == 0
    assert np.array_equal(ss.state(), st_w) and ss.accepted() == acc_w
    assert np.max(np.abs(series - np.asarray(series_w))) <= 2e-12 and abs(e - e_w) <= 2e-12
    assert np.array_equal(np.nan_to_num(ss.prediction(), nan=-1.0), np.nan_to_num(pred_w, nan=-1.0))


def test_peer_mode_temperature_matching_and_checks(mpr, inputs, slabs):
    values, mask, _ = inputs.make_rect_problem(96, 96, 8.0, 53, 0.66)
    g = mpr.Mpr(values, mask, mode="DP", seed=9)
    g.set_path("STRIP")
    T_w = g.estimate_temperature()[0]
    ss = slabs.make_slab_set(values, mask, 2, halo=4, mode="DP", seed=9, path="STRIP", peer=True)
    assert abs(ss.estimate_temperature() - T_w) <= 1e-9 * T_w and ss.exchanges == 0
    with pytest.raises(ValueError):
        slabs.make_slab_set(values, mask, 2, halo=8, mode="DP", seed=9, peer=True)
    # a context that is not a slab, or a neighbour that does not fit, is refused
    with pytest.raises(mpr.MprError):
        g.set_peers(None, ss.slabs[0].ctx)
    with pytest.raises(mpr.MprError):
        ss.slabs[0].ctx.set_peers(ss.slabs[1].ctx, None)       # slab 1 lies below slab 0, not above
    g.close()


def test_slab_without_measured_sites_of_its_own(mpr, slabs):
    """Sparse data on a thin grid: the rows of one slab hold no measured site at all, those of another a single value.
    The slab contexts are created all the same (mpr_create_slab), the range comes from the whole grid, and the result is
    the single context's."""
    Ly, Lx = 80, 6
    rng = np.random.default_rng(8)
    values = np.full((Ly, Lx), np.nan)
    mask = np.ones((Ly, Lx), dtype=np.uint8)
    for (y, x) in [(1, 2), (3, 4), (4, 4), (45, 1), (70, 3), (71, 3), (72, 0)]:       # rows 20..39 empty, rows 40..59 one value
        mask[y, x] = 0
        values[y, x] = rng.normal(50.0, 10.0)
    for mode, peer in (("DP", False), ("SP_INTRINSIC", True)):
        g = mpr.Mpr(values, mask, mode=mode, seed=4)
        g.set_path("STRIP"); g.set_temperature(0.3)
        pred, e, se = g.run(6, 3)
        st_w, acc_w = g.get_state().cpu().numpy(), g.counters()[0]
        g.close()
        ss = slabs.make_slab_set(values, mask, 4, halo=4, mode=mode, seed=4, path="STRIP", peer=peer)
        ss.set_temperature(0.3)
        ss.reset_chain(0)
        series, e_s, se_s = ss.run(6, 3)
        assert np.array_equal(ss.state(), st_w) and ss.accepted() == acc_w and abs(e_s - e) <= 2e-12
    # a context created for a slab is not usable before it is told its place
    h = mpr.Mpr(values[20:40], mask[20:40], slab=True)
    with pytest.raises(mpr.MprError) as ei:
        h.sweep(1)
    assert ei.value.code == mpr.ERR_NOT_READY
    # ... and the ordinary creation call still refuses such rows
    with pytest.raises(mpr.MprError) as ei:
        mpr.Mpr(values[20:40], mask[20:40])
    assert ei.value.code == mpr.ERR_NO_MEASURED


@pytest.mark.parametrize("mode,schedule,count", [("SP_INTRINSIC", "R4", 3), ("DP", "SITE_FUSED", 2), ("SP_INTRINSIC", "R4", 4)])
def test_peer_mode_with_a_stream_per_slab(mpr, inputs, slabs, mode, schedule, count):
    """Peer mode with every slab on a stream of its own: nothing but the events SlabSet records after each launch and
    waits for before the neighbours' next one orders the kernels (on one stream the stream order would).  Same spins as
    the single context, for runs long enough that unordered kernels would overlap."""
    Ly, Lx = 1100, 700
    values, mask, _ = inputs.make_rect_problem(Ly, Lx, 12.0, 57, 0.8)
    T, n_eq, n_meas = 0.02, 25, 5
    st_w, acc_w, series_w, pred_w, e_w, se_w, _, _ = whole(mpr, values, mask, mode, 79, "STRIP", schedule, T, n_eq, n_meas)
    ss = slabs.make_slab_set(values, mask, count, halo=4, mode=mode, seed=79, path="STRIP", schedule=schedule, peer=True,
                             streams=True)
    assert ss._own_streams and len({s.stream.cuda_stream for s in ss.slabs.values()}) == count
    ss.set_temperature(T)
    ss.reset_chain(0)
    series, e, se = ss.run(n_eq, n_meas)
    assert np.array_equal(ss.state(), st_w) and ss.accepted() == acc_w
    assert abs(e - e_w) <= 2e-12
    assert np.array_equal(np.nan_to_num(ss.prediction(), nan=-1.0), np.nan_to_num(pred_w, nan=-1.0))
