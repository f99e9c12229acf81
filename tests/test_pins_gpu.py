"""GPU-side checks that do not go through the oracle's copy of anything, plus the oracle comparison at
the headline size.

* the library's e_stderr against a numpy statement of R16 written here;
* a failed temperature estimate leaves no trial temperature behind;
* the two-step create (mpr_create without workspace, mpr_set_workspace, mpr_set_stream);
* launch geometry at the largest supported grid;
* the float-arithmetic moves (SP_PRECISE, SP_INTRINSIC: their own random-word mapping R9, ex2 / rcp forms)
  against the EXACT conditional density of PAPER.md Eq. 2 -- isolated free sites whose neighbours are
  all measured and identical from site to site, pooled over sites and sweeps, chi^2 by quadrature;
* DP against the oracle on the full L = 16384 grid of BASELINE.json configs[4]."""
import math

import numpy as np
import pytest

pytestmark = pytest.mark.gpu

TWO_PI = 2.0 * math.pi
PATHS = ["PLAIN", "TILED", "STRIP"]


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


# --------------------------------------------------------------------------- R16 on the library's own series
@pytest.mark.parametrize("n_meas", [7, 20, 53, 200])
def test_run_stderr_is_the_r16_binning(mpr, inputs, n_meas):
    values, mask, _ = inputs.make_problem(96, 8.0, 3, 0.66, False)
    g = mpr.Mpr(values, mask, mode="DP", seed=9)
    g.set_temperature(0.05)
    _, e, se = g.run(10, n_meas)
    v = g.series()
    assert len(v) == n_meas
    nb = 10 if n_meas >= 20 else n_meas
    ln = n_meas // nb
    bm = v[:nb * ln].reshape(nb, ln).mean(axis=1)
    assert abs(e - math.fsum(v) / n_meas) <= 1e-14
    assert abs(se - math.sqrt(bm.var(ddof=1) / nb)) <= 1e-9 * se + 1e-16
    assert se > 0.0


def test_failed_estimate_leaves_no_trial_temperature(mpr):
    L = 12
    z = np.where(np.arange(L)[None, :] < 6, 10.0, 20.0) * np.ones((L, 1))
    rng = np.random.default_rng(0)
    mask = np.zeros((L, L), dtype=np.uint8)
    mask[:, 5:7] = 1
    mask[rng.integers(0, L, 20), rng.integers(0, 4, 20)] = 1
    g = mpr.Mpr(z, mask, seed=2)
    with pytest.raises(mpr.MprError) as ei:
        g.estimate_temperature()
    assert ei.value.code == mpr.ERR_NO_ROOT
    with pytest.raises(mpr.MprError) as ei:          # T was never set: still not ready
        g.run(1, 1)
    assert ei.value.code == mpr.ERR_NOT_READY
    g.set_temperature(0.2)
    g.sweep(3)
    ref = g.get_state().cpu().numpy()
    cnt = g.counters()
    with pytest.raises(mpr.MprError):
        g.estimate_temperature()
    assert g.info()["T"] == 0.2                       # restored, and the chain restarts from trial 0
    g.sweep(3)
    assert np.array_equal(g.get_state().cpu().numpy(), ref) and g.counters() == cnt


def test_two_step_create_workspace_and_stream(mpr, inputs):
    import ctypes as C
    import torch
    values, mask, _ = inputs.make_problem(200, 10.0, 8, 0.66, False)
    dv, dm = torch.from_numpy(values).cuda(), torch.from_numpy(mask).cuda()
    ref = mpr.Mpr(dv, dm, mode="SP_INTRINSIC", seed=4)
    ref.set_temperature(0.03)
    ref.sweep(6)
    want = ref.get_state()
    lib = mpr.lib()
    h = C.c_void_p()
    assert lib.mpr_create(C.byref(h), 200, dv.data_ptr(), dm.data_ptr(), None, 0, None) == 0
    assert lib.mpr_set_precision(h, mpr.MODES["SP_INTRINSIC"]) == 0
    assert lib.mpr_set_seed(h, 4) == 0
    assert lib.mpr_set_temperature(h, 0.03) == 0
    assert lib.mpr_sweep(h, 1) == mpr.ERR_WORKSPACE              # nothing attached yet
    ws = torch.empty(mpr.workspace_bytes(200) + 256, dtype=torch.uint8, device="cuda")
    off = (-ws.data_ptr()) % 256
    assert lib.mpr_set_workspace(h, ws.data_ptr() + off + 8, ws.numel() - off - 8) == mpr.ERR_WORKSPACE   # misaligned
    assert lib.mpr_set_workspace(h, ws.data_ptr() + off, 1024) == mpr.ERR_WORKSPACE                       # too small
    assert lib.mpr_set_workspace(h, ws.data_ptr() + off, ws.numel() - off) == 0
    s2 = torch.cuda.Stream()
    assert lib.mpr_sweep(h, 3) == 0                               # on the default stream ...
    assert lib.mpr_set_stream(h, s2.cuda_stream) == 0             # ... waited for here
    assert lib.mpr_sweep(h, 3) == 0
    got = torch.empty_like(want)
    assert lib.mpr_get_state(h, got.data_ptr()) == 0
    s2.synchronize()
    assert torch.equal(got, want)
    lib.mpr_destroy(h)


@pytest.mark.parametrize("mode", ["DP", "SP_INTRINSIC"])
def test_launch_geometry_at_the_largest_grid(mpr, mode):
    """L = 32768 (kMaxL): chain reset (quench launches at fused depth 2), fused sweeps, a measuring sweep.
    Values are synthetic ramps generated on the device (8 GiB); the check is that every launch
    configuration is accepted and the state stays a valid one."""
    import torch
    L = 32768
    x = torch.arange(L, device="cuda", dtype=torch.float64)
    dv = (x[None, :] * 0.001 + x[:, None] * 0.002).contiguous()
    dm = ((torch.arange(L, device="cuda")[None, :] * 7 + torch.arange(L, device="cuda")[:, None] * 13) % 10 < 9)
    dm = dm.to(torch.uint8).contiguous()
    dm[0, 0] = 0
    for path in [p for p in ("TILED", "STRIP") if p in mpr.PATHS]:
        g = mpr.Mpr(dv, dm, mode=mode, seed=1)
        g.set_path(path)
        g.set_quench(4)
        g.set_temperature(0.01)
        g.set_fused_sweeps(2)
        g.sweep(2)
        g.set_fused_sweeps(1)
        _, e, _ = g.run(1, 1, want_pred=False)
        assert -2.0 <= e <= 0.0
        acc, att, sw = g.counters()
        assert sw == 4 and att == 4 * g.info()["n_free"] and 0 < acc < att
        g.close()
        del g
        torch.cuda.empty_cache()


# --------------------------------------------------------------------------- exact conditional density (Eq. 2)
def _exact_cdf_edges(nbr_phis, T, nbins):
    """Bin edges of equal probability under p(phi) ~ exp(sum_j cos[(phi - phi_j)/2] / T) on [0, 2pi]
    (Eq. 2 with q = 1/2, J = 1), by the trapezoidal rule on a fine grid."""
    x = np.linspace(0.0, TWO_PI, 400001)
    w = np.zeros_like(x)
    for p in nbr_phis:
        w += np.cos(0.5 * (x - p))
    w = np.exp((w - w.max()) / T)
    cdf = np.concatenate([[0.0], np.cumsum(0.5 * (w[1:] + w[:-1]) * np.diff(x))])
    cdf /= cdf[-1]
    edges = np.interp(np.arange(1, nbins) / nbins, cdf, x)
    return np.concatenate([[0.0], edges, [TWO_PI + 1e-9]])


def _chi2(samples, nbr_phis, T, nbins=40):
    edges = _exact_cdf_edges(nbr_phis, T, nbins)
    cnt, _ = np.histogram(samples, bins=edges)
    assert cnt.sum() == samples.size                    # every sample inside [0, 2pi]
    exp = samples.size / nbins
    return float(((cnt - exp) ** 2 / exp).sum())


def _isolated_grid(L, classes):
    """values (phi used directly as data, range anchored at 0 and 2pi), mask and the site lists per class.
    classes: name -> (list of (x, y) free sites, dict offset -> neighbour angle)."""
    rng = np.random.default_rng(12)
    z = rng.uniform(0.5, 5.5, (L, L))
    mask = np.zeros((L, L), dtype=np.uint8)
    assigned = {}
    for name, (sites, nb) in classes.items():
        for (x, y) in sites:
            mask[y, x] = 1
            for (dx, dy), ang in nb.items():
                xx, yy = x + dx, y + dy
                assert 0 <= xx < L and 0 <= yy < L, (name, x, y, dx, dy)
                assert assigned.get((xx, yy), ang) == ang, (name, xx, yy)
                assigned[(xx, yy)] = ang
                z[yy, xx] = ang
    for (x, y) in assigned:
        assert mask[y, x] == 0, "a fixed neighbour must be a measured site"
    # anchors of the R1 map: z_min = 0, z_max = 2pi  =>  phi = 2pi (z / 2pi), equal to z to 1 ulp
    free = np.argwhere(mask == 1)
    for (ax, ay), val in (((L - 1, L // 2), 0.0), ((L - 1, L // 2 + 2), TWO_PI)):
        assert mask[ay, ax] == 0 and (ax, ay) not in assigned
        z[ay, ax] = val
    # isolation: no two free sites are neighbours
    m = mask.astype(bool)
    assert not (m[:, 1:] & m[:, :-1]).any() and not (m[1:, :] & m[:-1, :]).any()
    return z, mask, free


NB4 = {(-1, 0): 1.3, (1, 0): 2.9, (0, -1): 0.4, (0, 1): 4.1}


@pytest.mark.parametrize("T", [0.01, 0.1, 1.0])
@pytest.mark.parametrize("path", ["TILED", "STRIP"])
@pytest.mark.parametrize("mode", ["SP_PRECISE", "SP_INTRINSIC", "DS_INTRINSIC", "SP", "DP"])
def test_interior_sites_sample_the_exact_conditional_density(mpr, mode, path, T):
    """39204 isolated free sites, each with the same four measured neighbours; after 60 hybrid sweeps, 26
    snapshots 6 sweeps apart: ~10^6 samples, chi^2 with 39 degrees of freedom against the exact density.
    P(chi^2_39 > 85) = 2.6e-5; a temperature off by 5 % gives chi^2 in the thousands (checked below)."""
    if path == "STRIP" and "STRIP" not in mpr.PATHS:
        pytest.skip("no STRIP path in this build")
    L = 596
    sites = [(x, y) for y in range(2, L - 2, 3) for x in range(1, L - 3, 3)]
    z, mask, _ = _isolated_grid(L, {"interior": (sites, NB4)})
    g = mpr.Mpr(z, mask, mode=mode, seed=31 + int(1000 * T))
    g.set_path(path)
    g.set_temperature(T)
    g.sweep(60)
    ys, xs = np.array([s[1] for s in sites]), np.array([s[0] for s in sites])
    snaps = []
    for _ in range(26):
        g.sweep(6)
        snaps.append(g.get_state().cpu().numpy()[ys, xs])
    samples = np.concatenate(snaps)
    assert samples.size > 1_000_000
    nb = list(NB4.values())
    c2 = _chi2(samples, nb, T)
    assert c2 < 85.0, (mode, T, c2)
    if mode == "SP_INTRINSIC" and path == "TILED":
        assert _chi2(samples, nb, 1.05 * T) > 400.0          # the test has the power to see a 5 % error in T
        assert _chi2(samples, [a + 0.01 for a in nb], T) > 400.0 or T >= 1.0   # ... or a 0.01 rad shift


@pytest.mark.parametrize("T", [0.02, 0.5])
@pytest.mark.parametrize("mode", ["SP_PRECISE", "SP_INTRINSIC"])
def test_edge_and_corner_sites_sample_the_exact_conditional_density(mpr, mode, T):
    """Open boundaries (R2): free sites on the top edge (3 neighbours) and in two corners (2 neighbours) of a
    small grid, sampled over many sweeps (one snapshot every 5 sweeps)."""
    L = 20
    top = [(x, 0) for x in range(1, L - 2, 3)]
    nb_top = {(-1, 0): 0.9, (1, 0): 2.2, (0, 1): 3.4}
    corners = [(0, L - 1), (L - 1, L - 1)]
    z, mask, _ = _isolated_grid(L, {
        "top": (top, nb_top),
        "corner_l": ([corners[0]], {(1, 0): 2.0, (0, -1): 3.1}),
        "corner_r": ([corners[1]], {(-1, 0): 2.0, (0, -1): 3.1}),
    })
    g = mpr.Mpr(z, mask, mode=mode, seed=77)
    g.set_temperature(T)
    g.sweep(100)
    n_snap = 12000
    tops, cors = np.empty((n_snap, len(top))), np.empty((n_snap, 2))
    ty, tx = np.array([s[1] for s in top]), np.array([s[0] for s in top])
    for i in range(n_snap):
        g.sweep(5)
        st = g.get_state().cpu().numpy()
        tops[i] = st[ty, tx]
        cors[i] = st[[L - 1, L - 1], [0, L - 1]]
    assert _chi2(tops.ravel(), list(nb_top.values()), T) < 85.0
    assert _chi2(cors.ravel(), [2.0, 3.1], T) < 85.0
    assert _chi2(cors.ravel(), [2.0, 3.1, 3.1], T) > 200.0      # a corner is not an edge site


# --------------------------------------------------------------------------- DP vs oracle at the headline size
@pytest.mark.parametrize("path", ["TILED", "STRIP"])
def test_dp_full_size_matches_oracle(mpr, oracle_mod, inputs, path):
    """BASELINE.json configs[4]: L = 16384, 90 % masked, the grid bench.py times.  R8 initialisation with 2
    quench double passes, then 2 hybrid sweeps at T = 1.1e-3 in DP: every one of the 2.7e8 spins within
    1e-9 of the oracle's, identical accepted-move count (~15 s of the oracle on all host threads)."""
    if path == "STRIP" and "STRIP" not in mpr.PATHS:
        pytest.skip("no STRIP path in this build")
    import torch
    c, values, mask, _ = inputs.make_config(5)
    o = oracle_mod.Oracle(values=values, mask=mask, seed=c.mpr_seed, threads=oracle_mod.threads_available(),
                          n_quench=2)
    o.set_temperature(1.1e-3)
    o.hybrid_sweeps(2)
    so = o.get_state()
    cnt_o = o.counters()
    e_o = o.energy()[1]
    del o
    g = mpr.Mpr(torch.from_numpy(values).cuda(), torch.from_numpy(mask).cuda(), mode="DP", seed=c.mpr_seed)
    g.set_path(path)
    g.set_quench(2)
    g.set_temperature(1.1e-3)
    g.sweep(2)
    sg = g.get_state().cpu().numpy()
    assert g.counters() == cnt_o
    assert abs(g.energy()[1] - e_o) <= 1e-10
    g.close()
    worst = 0.0
    for r in range(0, c.L, 1024):                       # blockwise: no third 2 GiB array
        worst = max(worst, float(np.max(np.abs(sg[r:r + 1024] - so[r:r + 1024]))))
    assert worst <= 1e-9, worst


# --------------------------------------------------------------------------- pass synchronisation, long run
@pytest.mark.parametrize("mode", ["DP", "SP", "SP_PRECISE", "SP_INTRINSIC"])
def test_pass_synchronisation_long_stress(mpr, inputs, mode):
    """2000 hybrid sweeps at the deepest fusion on a grid of several CTAs per SM, with a second stream keeping
    the SMs busy with an unrelated kernel (so that CTAs of the sweep kernel are descheduled and resumed at
    arbitrary points): final spins and accepted-move counts equal the one-launch-per-pass PLAIN path's.
    compute-sanitizer's racecheck is closed on this pool; this is evidence, not proof."""
    import torch
    L = 2048
    values, mask, _ = inputs.make_problem(L, 48.0, 9, 0.9, False)
    dv, dm = torch.from_numpy(values).cuda(), torch.from_numpy(mask).cuda()
    out = {}
    side = torch.cuda.Stream()
    junk = torch.randn(4096, 4096, device="cuda")
    for path, k in [("PLAIN", 1), ("TILED", 4)] + ([("STRIP", 2), ("STRIP", 1)] if "STRIP" in mpr.PATHS else []):
        g = mpr.Mpr(dv, dm, mode=mode, seed=555)
        g.set_path(path)
        g.set_fused_sweeps(k)
        g.set_temperature(0.02)
        for _ in range(20):
            if path != "PLAIN":
                with torch.cuda.stream(side):
                    for _ in range(4):
                        junk = torch.tanh(junk @ junk * 1e-4)
            g.sweep(100)
        out[(path, k)] = (g.get_state(), g.counters())
        side.synchronize()
        g.close()
    ref = out[("PLAIN", 1)]
    for key, (st, cnt) in out.items():
        assert cnt == ref[1], (mode, key)
        assert torch.equal(st, ref[0]), (mode, key, int((st != ref[0]).sum()))


def test_metropolis_decision_filter_is_exact(mpr):
    """the double-arithmetic modes decide u2 < exp(-dE/T) through a float filter and evaluate the double
    exponential only when the filter cannot decide.  On random moves and on moves built to sit on the edge -- u2 within a
    few ulps, 2^-24 .. 2^-12 relative, of exp(x); x around the -120 log 2 cut of the filter, at the underflow of exp, at 0
    and above; u2 = 0 and u2 = 1 - 2^-53; NaN -- the filtered decision equals the plain double one, and on ordinary moves
    the filter decides alone all but ~1e-4 of the time."""
    rng = np.random.default_rng(12)
    T = 0.37

    def words_of(u):                       # the two Philox words whose u53 is floor(u 2^53) 2^-53
        k = np.floor(np.clip(u, 0.0, 1.0 - 2.0 ** -53) * 2.0 ** 53).astype(np.uint64)
        hi, lo = (k >> np.uint64(26)).astype(np.uint64), (k & np.uint64((1 << 26) - 1)).astype(np.uint64)
        return np.stack([(hi << np.uint64(5)).astype(np.uint32), (lo << np.uint64(6)).astype(np.uint32)], axis=1)

    n = 1 << 20
    x = np.concatenate([-rng.exponential(2.0, n), rng.uniform(-800.0, 5.0, n), rng.uniform(-84.0, -82.0, n),
                        rng.uniform(-1e-6, 1e-6, n)])
    u = rng.uniform(size=x.size)
    # edge cases: u at exp(x) (1 + eps) for eps from a few ulps to the width of the filter's margin and beyond
    xe = -rng.exponential(3.0, n)
    eps = rng.choice([-1, 1], n) * 2.0 ** rng.uniform(-53, -10, n)
    ue = np.exp(xe) * (1.0 + eps)
    xs = np.array([0.0, -0.0, 1e-300, -1e-300, 3.0, -745.1, -745.3, -1e4, np.nan, -83.17, -83.18, -83.2, -120 * math.log(2.0)])
    us = np.array([0.0, 1.0 - 2.0 ** -53, 2.0 ** -24, 2.0 ** -25, 0.5])
    xg, ug = np.meshgrid(xs, us)
    X = np.concatenate([x, xe, xg.ravel()])
    U = np.concatenate([u, ue, ug.ravel()])
    out = mpr.debug_accept(words_of(U), X * T, T)          # -dE = x T
    filtered, plain, fast = out & 1, (out >> 1) & 1, (out >> 2) & 1
    assert np.array_equal(filtered, plain)
    # the plain device decision is itself the textbook one wherever double rounding cannot matter
    clear = np.abs(U[: x.size] - np.exp(np.minimum(X[: x.size], 0.0))) > 1e-9
    assert np.array_equal(plain[: x.size][clear], (U[: x.size] < np.exp(np.minimum(X[: x.size], 0.0)))[clear].astype(np.uint8))
    assert 1.0 - fast[:n].mean() < 3e-4                    # ordinary moves: the filter decides alone
    assert fast[x.size: x.size + n].mean() < 0.9           # the edge cases do reach the double evaluation


@pytest.mark.parametrize("path", ["PLAIN", "LIST", "TILED", "STRIP"])
@pytest.mark.parametrize("mode", ["DP", "SP_INTRINSIC"])
def test_nothing_to_predict(mpr, path, mode):
    """The empty problem: every site measured.  Every path runs (no zero-sized launch), nothing moves, no move is
    attempted, the chain energy is the sample energy, the prediction is the input."""
    L = 70
    rng = np.random.default_rng(4)
    z = rng.normal(50.0, 10.0, (L, L))
    g = mpr.Mpr(z, np.zeros((L, L), dtype=np.uint8), mode=mode, seed=1)
    g.set_path(path)
    g.set_temperature(0.1)
    st0 = g.get_state().cpu().numpy()
    pred, e, se = g.run(3, 4)
    assert np.array_equal(g.get_state().cpu().numpy(), st0)
    assert g.counters() == (0, 0, 7)
    es, n_pairs = g.sample_energy()
    assert n_pairs == 2 * L * (L - 1) and abs(e - es) <= (1e-12 if mode == "DP" else 2e-6) and se <= 1e-12
    assert np.array_equal(pred.cpu().numpy(), z)
    for sched in ("SITE_FUSED",):
        if path != "TILED":
            g.set_schedule(sched)
            g.sweep(2)
            assert np.array_equal(g.get_state().cpu().numpy(), st0)
    g.close()


def test_one_prediction_site(mpr, oracle_mod):
    """The smallest non-empty problem on every path: one free site in a corner of a grid that is not a multiple of anything."""
    L = 67
    rng = np.random.default_rng(6)
    z = rng.normal(50.0, 10.0, (L, L))
    mask = np.zeros((L, L), dtype=np.uint8)
    mask[L - 1, L - 1] = 1
    o = oracle_mod.Oracle(values=z, mask=mask, seed=3)
    o.set_temperature(0.2)
    o.hybrid_sweeps(25)
    for path in ("PLAIN", "LIST", "TILED", "STRIP"):
        g = mpr.Mpr(z, mask, seed=3)
        g.set_path(path)
        g.set_temperature(0.2)
        g.sweep(25)
        assert np.max(np.abs(g.get_state().cpu().numpy() - o.get_state())) <= 1e-9, path
        assert g.counters() == o.counters(), path
        g.close()


def test_maximum_size_runs_and_paths_agree(mpr):
    """L = 32768, the largest grid the library accepts (2^30 sites; ~70 GB of workspace and inputs): STRIP (what AUTO picks),
    TILED and the per-pass kernels give the same spins after a chain reset and two sweeps, bit for bit -- no index
    arithmetic overflows anywhere on the way -- and the bookkeeping (prediction sites, attempted moves) is exact."""
    import torch
    dev = torch.device("cuda:0")
    if torch.cuda.mem_get_info(dev)[0] < 110 * 2 ** 30:
        pytest.skip("needs ~110 GB of free device memory")
    L = 32768
    gen = torch.Generator(device=dev)
    gen.manual_seed(17)
    # a smooth field plus noise, built on the device (the FFT recipe of inputs.py would need ~50 GB of host memory here)
    y = torch.arange(L, device=dev, dtype=torch.float64)
    values = 50.0 + 8.0 * torch.sin(y[:, None] * 3e-4) * torch.cos(y[None, :] * 2e-4)
    values += torch.randn((L, L), generator=gen, device=dev, dtype=torch.float64)
    mask = (torch.rand((L, L), generator=gen, device=dev) < 0.9).to(torch.uint8)
    n_free = int(mask.sum().item())
    ref = None
    for path in ("PLAIN", "STRIP", "TILED"):
        g = mpr.Mpr(values, mask, mode="SP_INTRINSIC", seed=23, device=dev)
        g.set_path(path)
        g.set_quench(2)
        g.set_temperature(0.002)
        g.sweep(2)
        assert g.info()["n_free"] == n_free
        acc, att, sw = g.counters()
        assert (att, sw) == (2 * n_free, 2) and 0 < acc < att
        st = g.get_state()
        H, e = g.energy()
        g.close()
        del g
        if ref is None:
            ref = (st, acc, e)
        else:
            assert torch.equal(st, ref[0]) and acc == ref[1], path
            assert abs(e - ref[2]) <= 1e-9
        del st
        torch.cuda.empty_cache()


def test_over_relaxation_tie_at_the_edge_of_the_range(mpr, oracle_mod):
    """A degenerate case with two valid outcomes (found by fuzzing 1 x n grids): in a chain of free sites next to a
    measured site at phi = 0 the quench passes leave exact relations such as phi_1 = phi_0 + phi_2, and the reflection
    phi' = phi_0 + phi_2 - phi_1 of R5 then lands on the edge of [0, 2 pi] to within rounding.  The oracle, working on
    angles, gets phi' = 0 and keeps it; the library, working on unit vectors, gets sin(q phi') = -1e-17 and leaves the
    spin -- "unchanged if phi' is outside [0, 2 pi]".  Both follow R5; which one happens is decided by the last bit.
    The test pins that this IS such a tie: up to the pass in question the two agree to rounding, the oracle's new angle
    is 0 within 1e-15, the library's spin is the old one, and the sum rule that produced the tie holds to rounding."""
    values = np.array([np.nan, np.nan, np.nan, 34.75851636, np.nan, 50.36306022, np.nan, np.nan]).reshape(8, 1)
    mask = np.isnan(values).astype(np.uint8)
    o = oracle_mod.Oracle(values=values, mask=mask, seed=5)
    g = mpr.Mpr(values, mask, mode="DP", seed=5)
    for h in (o, g):
        h.set_quench(4)
        h.set_temperature(0.3)
    g.set_path("PLAIN")
    for kind, c in [("MET", 0), ("MET", 1), ("OR", 0)]:
        if kind == "MET":
            o.met_pass(c, 1)
        else:
            o.or_pass(c)
        g.pass_(kind, c, 1)
    before_g, before_o = g.get_state().cpu().numpy().ravel(), o.get_state().ravel()
    assert np.max(np.abs(before_g - before_o)) <= 1e-15
    assert abs(before_o[0] + before_o[2] - before_o[1]) <= 1e-15          # the exact relation behind the tie
    o.or_pass(1)
    g.pass_("OR", 1, 1)
    after_g, after_o = g.get_state().cpu().numpy().ravel(), o.get_state().ravel()
    if abs(after_g[1] - after_o[1]) > 1e-12:                               # the tie went two ways (it does on B200 today)
        assert abs(after_o[1]) <= 1e-15 and after_g[1] == before_g[1]
    others = [i for i in range(8) if i != 1]
    assert np.max(np.abs(after_g[others] - after_o[others])) <= 1e-15
