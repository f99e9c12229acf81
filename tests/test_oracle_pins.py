"""Pins of the CPU oracle against what the paper and the mathematics fix.

None of these compares the oracle with itself or with the CUDA path: each expected value is
a closed form, an invariant, a brute-force sum, a quadrature of the exact Boltzmann density,
or a library routine (the CUDA toolkit's Philox block function).
"""
import ctypes as C
import json
import math
import os
import subprocess

import numpy as np
import pytest
from scipy import stats

HERE = os.path.dirname(os.path.abspath(__file__))
TWO_PI = 2.0 * math.pi
Q = 0.5

with open(os.path.join(HERE, "golden", "closed_forms.json")) as fh:
    CLOSED = json.load(fh)


def grid_with_free(L, free_sites, phi):
    mask = np.zeros((L, L), dtype=np.uint8)
    for (x, y) in free_sites:
        mask[y, x] = 1
    return mask, np.array(phi, dtype=np.float64).reshape(L, L)


# --------------------------------------------------------------------------- Philox (T8)
@pytest.fixture(scope="module")
def curand_ref():
    src = os.path.join(HERE, "helpers", "curand_philox_host.cu")
    so = os.path.join(HERE, "helpers", "libcurand_philox_host.so")
    if not os.path.exists(so) or os.path.getmtime(so) < os.path.getmtime(src):
        subprocess.run(["nvcc", "-O2", "-shared", "-Xcompiler", "-fPIC", "-Wno-deprecated-gpu-targets",
                        "-o", so, src], check=True)
    lib = C.CDLL(so)
    u32p = C.POINTER(C.c_uint32)
    lib.ref_philox4x32_10.argtypes = [u32p, u32p, u32p]

    def ref(ctr, key):
        c = (C.c_uint32 * 4)(*ctr)
        k = (C.c_uint32 * 2)(*key)
        o = (C.c_uint32 * 4)()
        lib.ref_philox4x32_10(c, k, o)
        return [int(v) for v in o]
    return ref


def test_philox_matches_cuda_toolkit(oracle_mod, curand_ref):
    rng = np.random.default_rng(123)
    cases = [([0, 0, 0, 0], [0, 0]), ([0xFFFFFFFF] * 4, [0xFFFFFFFF] * 2), ([1, 2, 3, 4], [5, 6])]
    for _ in range(2000):
        cases.append(([int(v) for v in rng.integers(0, 2 ** 32, 4)], [int(v) for v in rng.integers(0, 2 ** 32, 2)]))
    for ctr, key in cases:
        assert oracle_mod.philox4x32_10(ctr, key) == curand_ref(ctr, key)


def test_philox_constants_match_toolkit_header():
    """The four constants the oracle restates are the ones in the toolkit header (SURVEY 8c note)."""
    hdr = "/usr/local/cuda/include/curand_philox4x32_x.h"
    if not os.path.exists(hdr):
        pytest.skip("CUDA toolkit header not present")
    text = open(hdr).read()
    src = open(os.path.join(os.path.dirname(HERE), "oracle", "mpr_oracle.cpp")).read()
    for name in ("PHILOX_W32_0", "PHILOX_W32_1", "PHILOX_M4x32_0", "PHILOX_M4x32_1"):
        val = int(text.split("#define " + name)[1].split("(")[1].split(")")[0].strip(), 16)
        assert ("0x%08x" % val) in src.lower(), name


def test_u53_exact(oracle_mod):
    rng = np.random.default_rng(5)
    assert oracle_mod.u53(0, 0) == 0.0
    assert oracle_mod.u53(0xFFFFFFFF, 0xFFFFFFFF) == 1.0 - 2.0 ** -53
    for _ in range(1000):
        a, b = (int(v) for v in rng.integers(0, 2 ** 32, 2))
        expect = (((a >> 5) << 26) | (b >> 6)) / float(2 ** 53)
        assert oracle_mod.u53(a, b) == expect


def test_init_is_uniform(oracle_mod):
    """O2: free spins i.i.d. uniform on [0, 2pi): KS test + lag-1 correlation on 65536 sites."""
    L = 256
    mask = np.ones((L, L), dtype=np.uint8)
    o = oracle_mod.Oracle(phi=np.zeros((L, L)), mask=mask)
    o.init_random(trial=0)
    phi = o.get_state().ravel()
    assert phi.min() >= 0.0 and phi.max() < TWO_PI
    assert stats.kstest(phi / TWO_PI, "uniform").pvalue > 1e-3
    r = np.corrcoef(phi[:-1], phi[1:])[0, 1]
    assert abs(r) < 4.0 / math.sqrt(phi.size)
    o.init_random(trial=1)
    phi1 = o.get_state().ravel()
    assert abs(np.corrcoef(phi, phi1)[0, 1]) < 4.0 / math.sqrt(phi.size)


# --------------------------------------------------------------------------- energy (T1, T2)
def test_ground_state_energy(oracle_mod):
    """Uniform grid => every bond contributes -J, e = 2H/N_b = -2J exactly (closed form)."""
    for L in (2, 3, 8, 33):
        mask = np.zeros((L, L), dtype=np.uint8)
        o = oracle_mod.Oracle(phi=np.full((L, L), 1.2345), mask=mask)
        H, e = o.energy()
        assert e == CLOSED["e_ground_state"]["value"]
        assert H == -2.0 * L * (L - 1)


def test_infinite_temperature_energy_static(oracle_mod):
    """i.i.d. uniform spins: E[e] = -2J (2/pi)^2 = -8/pi^2, Var[cos] = 1/2 - 16/pi^4."""
    L = 256
    o = oracle_mod.Oracle(phi=np.zeros((L, L)), mask=np.ones((L, L), dtype=np.uint8))
    o.init_random(0)
    _, e = o.energy()
    nb = 2 * L * (L - 1)
    se = 2.0 * math.sqrt((0.5 - 16.0 / math.pi ** 4) / nb)
    expect = CLOSED["e_infinite_temperature"]["value"]
    assert abs(expect - (-8.0 / math.pi ** 2)) < 1e-12
    assert abs(e - expect) < 4.0 * se


def test_infinite_temperature_energy_dynamic(oracle_mod):
    """All sites free, T = 1e6: the hybrid chain samples the uniform measure, e -> -8/pi^2."""
    L = 48
    o = oracle_mod.Oracle(phi=np.full((L, L), 3.0), mask=np.ones((L, L), dtype=np.uint8))
    o.set_seed(77)
    o.set_quench(0)
    o.set_temperature(1e6)
    o.hybrid_sweeps(50)
    es = o.trace_energy(400)
    m, se = oracle_mod.mean_stderr(es)
    assert abs(m - CLOSED["e_infinite_temperature"]["value"]) < 4.0 * se + 1e-4
    acc, att, _ = o.counters()
    assert att == 450 * L * L


def brute_force_H(phi):
    L = phi.shape[0]
    ys, xs = np.mgrid[0:L, 0:L]
    xs, ys, p = xs.ravel(), ys.ravel(), phi.ravel()
    H = 0.0
    for i in range(p.size):
        for j in range(i + 1, p.size):
            if abs(xs[i] - xs[j]) + abs(ys[i] - ys[j]) == 1:
                H -= math.cos(Q * (p[i] - p[j]))
    return H


def test_energy_vs_brute_force(oracle_mod):
    rng = np.random.default_rng(1)
    for L in (2, 3, 5, 8):
        phi = rng.uniform(0, TWO_PI, (L, L))
        o = oracle_mod.Oracle(phi=phi, mask=np.zeros((L, L), dtype=np.uint8))
        H, e = o.energy()
        Hb = brute_force_H(phi)
        assert abs(H - Hb) < 1e-12 * max(1.0, abs(Hb))
        assert abs(e - 2.0 * Hb / (2 * L * (L - 1))) < 1e-13


def test_local_energy_is_site_part_of_H(oracle_mod):
    """H(phi with site s changed) - H(phi) == E_loc(new) - E_loc(old): includes edges and corners."""
    rng = np.random.default_rng(2)
    L = 5
    phi = rng.uniform(0, TWO_PI, (L, L))
    o = oracle_mod.Oracle(phi=phi, mask=np.zeros((L, L), dtype=np.uint8))
    H0 = brute_force_H(phi)
    for (x, y) in [(0, 0), (4, 0), (0, 4), (4, 4), (2, 0), (0, 2), (2, 2), (3, 1)]:
        new = rng.uniform(0, TWO_PI)
        p2 = phi.copy()
        p2[y, x] = new
        d = o.local_energy(x, y, new) - o.local_energy(x, y, phi[y, x])
        assert abs((brute_force_H(p2) - H0) - d) < 1e-12


def test_sample_energy_counts_measured_pairs_only(oracle_mod):
    rng = np.random.default_rng(3)
    L = 7
    phi = rng.uniform(0, TWO_PI, (L, L))
    mask = (rng.uniform(size=(L, L)) < 0.4).astype(np.uint8)
    o = oracle_mod.Oracle(phi=phi, mask=mask)
    es, n = o.sample_energy()
    tot, cnt = 0.0, 0
    for y in range(L):
        for x in range(L):
            for (dx, dy) in ((1, 0), (0, 1)):
                X, Y = x + dx, y + dy
                if X < L and Y < L and not mask[y, x] and not mask[Y, X]:
                    tot += math.cos(Q * (phi[y, x] - phi[Y, X]))
                    cnt += 1
    assert n == cnt
    assert abs(es - (-2.0 * tot / cnt)) < 1e-13
    # all measured and uniform => e_s = -2 (same normalisation as e)
    o2 = oracle_mod.Oracle(phi=np.full((L, L), 0.7), mask=np.zeros((L, L), dtype=np.uint8))
    assert o2.sample_energy() == (-2.0, 2 * L * (L - 1))


# --------------------------------------------------------------------------- over-relaxation (T3)
def test_over_relaxation_conserves_local_energy(oracle_mod):
    """|E_loc(phi') - E_loc(phi)| <= 1e-12 for interior, edge and corner sites (R5)."""
    rng = np.random.default_rng(4)
    L = 3
    worst, moved = 0.0, 0
    for trial in range(4000):
        phi = rng.uniform(0, TWO_PI, (L, L))
        x, y = [(1, 1), (0, 0), (1, 0), (2, 1), (2, 2)][trial % 5]
        mask = np.zeros((L, L), dtype=np.uint8)
        mask[y, x] = 1
        o = oracle_mod.Oracle(phi=phi, mask=mask)
        e0 = o.local_energy(x, y, phi[y, x])
        o.or_pass((x + y) & 1)
        new = o.get_state()[y, x]
        assert 0.0 <= new <= TWO_PI
        if new != phi[y, x]:
            moved += 1
            worst = max(worst, abs(o.local_energy(x, y, new) - e0))
            # closed form of the reflection: q phi' = 2 Phi - q phi
            nb = [(x - 1, y), (x + 1, y), (x, y - 1), (x, y + 1)]
            nb = [(a, b) for a, b in nb if 0 <= a < L and 0 <= b < L]
            A = sum(math.cos(Q * phi[b, a]) for a, b in nb)
            B = sum(math.sin(Q * phi[b, a]) for a, b in nb)
            assert abs(new - (2.0 * math.atan2(B, A) / Q - phi[y, x])) < 1e-12
    assert moved > 2000
    assert worst <= 1e-12


def test_over_relaxation_conserves_H_and_is_involution(oracle_mod):
    rng = np.random.default_rng(6)
    L = 24
    # smooth-ish field so that most reflections stay in range
    phi = np.clip(3.0 + 0.5 * rng.standard_normal((L, L)), 0, TWO_PI)
    o = oracle_mod.Oracle(phi=phi, mask=np.ones((L, L), dtype=np.uint8))
    H0, _ = o.energy()
    for c in (0, 1, 0, 1):
        o.or_pass(c)
        H1, _ = o.energy()
        assert abs(H1 - H0) < 1e-10
    o.set_state(phi)
    o.or_pass(0)
    once = o.get_state()
    assert np.mean(once != phi) > 0.3
    o.or_pass(0)
    twice = o.get_state()
    # a reflection that stayed in range is undone by the second one
    assert np.max(np.abs(twice - phi)) < 1e-12


def test_over_relaxation_rejects_out_of_range(oracle_mod):
    """phi' = 2 Phi/q - phi outside [0, 2pi] must leave the spin unchanged (R5)."""
    L = 3
    phi = np.full((L, L), 0.2)
    phi[1, 1] = 3.0          # reflection about ~0.2 gives -2.6 < 0
    mask = np.zeros((L, L), dtype=np.uint8)
    mask[1, 1] = 1
    o = oracle_mod.Oracle(phi=phi, mask=mask)
    o.or_pass(0)
    assert o.get_state()[1, 1] == 3.0


# --------------------------------------------------------------------------- Metropolis / hybrid (T4, T5)
def exact_density_cdf(nbr_phis, T, n=400001):
    x = np.linspace(0.0, TWO_PI, n)
    logw = sum(np.cos(Q * (x - pj)) for pj in nbr_phis) / T
    w = np.exp(logw - logw.max())
    cdf = np.concatenate([[0.0], np.cumsum(0.5 * (w[1:] + w[:-1]) * np.diff(x))])
    Z = cdf[-1]
    return x, w / Z, cdf / Z


def chi2_against_density(samples, nbr_phis, T, nbins=50):
    x, _, cdf = exact_density_cdf(nbr_phis, T)
    edges = np.interp(np.linspace(0, 1, nbins + 1), cdf, x)
    edges[0], edges[-1] = 0.0, TWO_PI
    counts, _ = np.histogram(samples, bins=edges)
    assert counts.sum() == samples.size            # every sample inside [0, 2pi]
    expected = samples.size / nbins
    chi2 = float(np.sum((counts - expected) ** 2 / expected))
    return chi2, stats.chi2.sf(chi2, nbins - 1)


SITE_CASES = [
    # (free site, neighbour phis written at left,right,up,down where they exist)
    ((1, 1), {(0, 1): 1.0, (2, 1): 2.5, (1, 0): 4.0, (1, 2): 0.3}),
    ((0, 0), {(1, 0): 5.5, (0, 1): 4.4}),
    ((1, 0), {(0, 0): 0.4, (2, 0): 1.1, (1, 1): 2.0}),
]


@pytest.mark.parametrize("kind", [0, 1, 2], ids=["metropolis", "hybrid", "hybrid-site-fused"])
@pytest.mark.parametrize("T", [0.01, 0.1, 1.0, 10.0])
@pytest.mark.parametrize("case", [0, 1, 2], ids=["interior4", "corner2", "edge3"])
def test_single_site_histogram(oracle_mod, kind, T, case):
    """10^6 thinned draws at one free site with fixed neighbours vs p(phi) ~ exp(sum_j cos[q(phi-phi_j)]/T).
    kind 2 = hybrid sweeps in the site-fused pass order R4b (MET c0, OR c0, MET c1, OR c1)."""
    (x, y), nbrs = SITE_CASES[case]
    L = 3
    phi = np.full((L, L), 3.0)
    for (a, b), v in nbrs.items():
        phi[b, a] = v
    mask = np.zeros((L, L), dtype=np.uint8)
    mask[y, x] = 1
    o = oracle_mod.Oracle(phi=phi, mask=mask)
    o.set_quench(0)
    o.set_seed(1234 + 17 * case + kind)
    o.set_temperature(T)
    if kind == 2:
        o.set_schedule("SITE_FUSED")
    thin = 8
    tr = o.trace(1_000_000 * thin // 4, min(kind, 1), [y * L + x])[:, 0]
    samples = tr[1000::thin]
    chi2, p = chi2_against_density(samples, list(nbrs.values()), T)
    assert p > 1e-4, (chi2, p)
    # measured neighbours never move
    st = o.get_state()
    for (a, b), v in nbrs.items():
        assert st[b, a] == v


def test_histogram_detects_a_wrong_temperature(oracle_mod):
    """Power check of the chi^2 pin: the same samples fail against the density at 1.15 T."""
    (x, y), nbrs = SITE_CASES[0]
    L = 3
    phi = np.full((L, L), 3.0)
    for (a, b), v in nbrs.items():
        phi[b, a] = v
    mask = np.zeros((L, L), dtype=np.uint8)
    mask[y, x] = 1
    o = oracle_mod.Oracle(phi=phi, mask=mask)
    o.set_quench(0)
    o.set_seed(99)
    o.set_temperature(0.1)
    tr = o.trace(2_000_000, 0, [y * L + x])[1000::8, 0]
    assert chi2_against_density(tr, list(nbrs.values()), 0.1)[1] > 1e-4
    assert chi2_against_density(tr, list(nbrs.values()), 0.115)[1] < 1e-6


# --------------------------------------------------------------------------- two free sites (T6)
@pytest.mark.parametrize("schedule", ["R4", "SITE_FUSED"])
def test_two_free_sites_vs_quadrature(oracle_mod, schedule):
    """Two neighbouring free sites (one of each colour) in a ring of fixed spins: the chain's means against a 2-D
    quadrature of the Boltzmann weight.  In the site-fused order the over-relaxation move of site a uses site b
    BEFORE b's Metropolis move of the same sweep: a wrong composition shows here."""
    rng = np.random.default_rng(8)
    L = 4
    phi = rng.uniform(0.5, 5.5, (L, L))
    mask = np.zeros((L, L), dtype=np.uint8)
    mask[1, 1] = mask[1, 2] = 1
    T = 0.3
    o = oracle_mod.Oracle(phi=phi, mask=mask)
    o.set_quench(0)
    o.set_seed(4242)
    o.set_temperature(T)
    o.set_schedule(schedule)
    tr = o.trace(800_000, 1, [1 * L + 1, 1 * L + 2])[2000:]
    # exact: p(a,b) ~ exp{[sum_fixed-nbrs cos(q(a-.)) + sum cos(q(b-.)) + cos(q(a-b))]/T}
    n = 1201
    g = np.linspace(0, TWO_PI, n)
    wq = np.full(n, g[1] - g[0]); wq[0] *= 0.5; wq[-1] *= 0.5
    fa = sum(np.cos(Q * (g - phi[yy, xx])) for (xx, yy) in [(0, 1), (1, 0), (1, 2)])
    fb = sum(np.cos(Q * (g - phi[yy, xx])) for (xx, yy) in [(3, 1), (2, 0), (2, 2)])
    logw = (fa[:, None] + fb[None, :] + np.cos(Q * (g[:, None] - g[None, :]))) / T
    w = np.exp(logw - logw.max()) * wq[:, None] * wq[None, :]
    w /= w.sum()
    exact = {
        "a": float((w.sum(1) * g).sum()),
        "b": float((w.sum(0) * g).sum()),
        "cab": float((w * np.cos(Q * (g[:, None] - g[None, :]))).sum()),
    }
    obs = {"a": tr[:, 0], "b": tr[:, 1], "cab": np.cos(Q * (tr[:, 0] - tr[:, 1]))}
    for k in exact:
        v = obs[k]
        nb = 100
        bm = v[: (v.size // nb) * nb].reshape(nb, -1).mean(1)
        se = bm.std(ddof=1) / math.sqrt(nb)
        assert abs(v.mean() - exact[k]) < 4.0 * se, (k, v.mean(), exact[k], se)


# --------------------------------------------------------------------------- limits (T7), equipartition
def test_zero_temperature_limit_single_site(oracle_mod):
    (x, y), nbrs = SITE_CASES[0]
    L = 3
    phi = np.full((L, L), 3.0)
    for (a, b), v in nbrs.items():
        phi[b, a] = v
    phi[y, x] = 6.0
    mask = np.zeros((L, L), dtype=np.uint8)
    mask[y, x] = 1
    A = sum(math.cos(Q * v) for v in nbrs.values())
    B = sum(math.sin(Q * v) for v in nbrs.values())
    star = math.atan2(B, A) / Q
    T = 1e-8
    o = oracle_mod.Oracle(phi=phi, mask=mask)
    o.set_quench(0)
    o.set_seed(5)
    o.set_temperature(T)
    tr = o.trace(400_000, 1, [y * L + x])[:, 0]
    assert abs(tr[-20000:].mean() - star) < 5e-5          # thermal width sqrt(T/R q^2) ~ 1e-4
    # and the quench pass lands on the minimiser at once
    o2 = oracle_mod.Oracle(phi=phi, mask=mask)
    o2.quench_pass((x + y) & 1)
    assert abs(o2.get_state()[y, x] - star) < 1e-14


def test_quench_never_raises_energy_and_stays_in_range(oracle_mod):
    rng = np.random.default_rng(10)
    L = 40
    phi = rng.uniform(0, TWO_PI, (L, L))
    mask = (rng.uniform(size=(L, L)) < 0.8).astype(np.uint8)
    o = oracle_mod.Oracle(phi=phi, mask=mask)
    H_prev, _ = o.energy()
    for k in range(20):
        for c in (0, 1):
            o.quench_pass(c)
            H, _ = o.energy()
            assert H <= H_prev + 1e-9
            H_prev = H
    st = o.get_state()
    assert st.min() >= 0.0 and st.max() <= TWO_PI
    assert np.array_equal(st[mask == 0], phi[mask == 0])


def test_equipartition_slope(oracle_mod):
    """Low-T harmonic limit: one quadratic degree of freedom per free site => d e/dT -> (f/2) N/(N_b/2)."""
    from paper_1910_08448_b200 import inputs
    values, mask, _ = inputs.make_problem(64, 8.0, 0, 0.33)
    o = oracle_mod.Oracle(values=values, mask=mask, seed=1000)
    e1, s1 = o.trial_energy(0.01, 1)
    e2, s2 = o.trial_energy(0.03, 2)
    f = mask.mean()
    slope = (e2 - e1) / 0.02
    expect = 0.5 * f * 64.0 / 63.0
    assert abs(slope / expect - 1.0) < 0.05, (slope, expect)


# --------------------------------------------------------------------------- mapping, invariants (T9)
def test_mapping_round_trip_and_errors(oracle_mod):
    rng = np.random.default_rng(11)
    L = 16
    z = rng.normal(50, 10, (L, L))
    mask = (rng.uniform(size=(L, L)) < 0.5).astype(np.uint8)
    vals = z.copy()
    vals[mask == 1] = np.nan
    o = oracle_mod.Oracle(values=vals, mask=mask, seed=3)
    zmin, zmax = o.zrange()
    assert zmin == z[mask == 0].min() and zmax == z[mask == 0].max()
    phi = o.get_state()
    np.testing.assert_allclose(phi[mask == 0], TWO_PI * (z[mask == 0] - zmin) / (zmax - zmin), rtol=0, atol=1e-15)
    assert phi[mask == 0].min() == 0.0 and phi[mask == 0].max() == TWO_PI
    o.set_temperature(0.05)
    pred, e, se = o.run(5, 10)
    assert np.array_equal(pred[mask == 0], z[mask == 0])              # bit-exact at measured sites
    assert pred[mask == 1].min() >= zmin - 1e-12 and pred[mask == 1].max() <= zmax + 1e-12
    # measured spins are never touched; all spins stay in [0, 2pi]
    st = o.get_state()
    assert np.array_equal(st[mask == 0], phi[mask == 0])
    assert st.min() >= 0.0 and st.max() <= TWO_PI
    # error paths
    for bad_vals, bad_mask, code in [
        (vals, np.ones((L, L), dtype=np.uint8), oracle_mod.ERR_NO_MEASURED),
        (np.full((L, L), 3.0), np.zeros((L, L), dtype=np.uint8), oracle_mod.ERR_DEGENERATE_RANGE),
        (np.where(mask == 1, 1.0, np.inf), mask, oracle_mod.ERR_NONFINITE),
    ]:
        with pytest.raises(oracle_mod.OracleError) as ei:
            oracle_mod.Oracle(values=bad_vals, mask=bad_mask)
        assert ei.value.code == code
    o3 = oracle_mod.Oracle(values=vals, mask=mask)
    with pytest.raises(oracle_mod.OracleError) as ei:
        o3.run(1, 1)                                                    # T not set
    assert ei.value.code == oracle_mod.ERR_NOT_READY


def test_constant_neighbourhood_predicts_the_constant(oracle_mod):
    """A free site whose whole neighbourhood holds one value is predicted at that value as T -> 0."""
    L = 16
    z = np.where(np.arange(L)[None, :] < 8, 10.0, 20.0) * np.ones((L, 1))
    mask = np.zeros((L, L), dtype=np.uint8)
    mask[8, 2] = mask[5, 12] = 1
    vals = z.copy()
    vals[mask == 1] = np.nan
    o = oracle_mod.Oracle(values=vals, mask=mask, seed=1)
    o.set_temperature(1e-6)
    pred, _, _ = o.run(50, 200)
    assert abs(pred[8, 2] - 10.0) < 0.02
    assert abs(pred[5, 12] - 20.0) < 0.02


def test_sweep_order_and_chain_continuation(oracle_mod):
    """R4: a hybrid sweep is MET(0), MET(1), OR(0), OR(1) with the sweep number in the Philox counter;
    run(a,0) then run(0,b) equals run(a,b)."""
    from paper_1910_08448_b200 import inputs
    values, mask, _ = inputs.make_problem(32, 6.0, 7, 0.6)
    a = oracle_mod.Oracle(values=values, mask=mask, seed=9)
    b = oracle_mod.Oracle(values=values, mask=mask, seed=9)
    a.set_temperature(0.05); b.set_temperature(0.05)
    a.hybrid_sweeps(3)
    for n in (1, 2, 3):
        b.met_pass(0, n); b.met_pass(1, n); b.or_pass(0); b.or_pass(1)
    assert np.array_equal(a.get_state(), b.get_state())
    c = oracle_mod.Oracle(values=values, mask=mask, seed=9)
    d = oracle_mod.Oracle(values=values, mask=mask, seed=9)
    c.set_temperature(0.05); d.set_temperature(0.05)
    p1, e1, s1 = c.run(4, 6)
    d.run(4, 0)
    p2, e2, s2 = d.run(0, 6)
    assert np.array_equal(p1, p2) and e1 == e2 and s1 == s2
    # a different seed gives a different chain
    e_ = oracle_mod.Oracle(values=values, mask=mask, seed=10)
    e_.set_temperature(0.05)
    e_.hybrid_sweeps(3)
    assert not np.array_equal(a.get_state(), e_.get_state())
    # threads change nothing (counter-based generator)
    t = oracle_mod.Oracle(values=values, mask=mask, seed=9, threads=3)
    t.set_temperature(0.05)
    t.hybrid_sweeps(3)
    assert np.array_equal(a.get_state(), t.get_state())
    assert a.counters() == t.counters()


def test_mean_stderr_binning(oracle_mod):
    rng = np.random.default_rng(12)
    ses = []
    for _ in range(100):
        v = rng.normal(3.0, 2.0, 1000)
        m, se = oracle_mod.mean_stderr(v)
        assert abs(m - v.mean()) < 1e-12
        ses.append(se)
    # i.i.d. data: the binned error estimates sigma/sqrt(n) (10 bins => ~24 % scatter per estimate)
    assert abs(np.mean(ses) / (2.0 / math.sqrt(1000)) - 1.0) < 0.1
    # positively correlated series: the binned error must exceed the naive one
    w = np.convolve(rng.normal(0, 1, 5000), np.ones(50) / 50, mode="valid")
    _, se_w = oracle_mod.mean_stderr(w)
    assert se_w > 2.0 * w.std(ddof=1) / math.sqrt(w.size)
    assert oracle_mod.mean_stderr([1.0])[1] == 0.0


# --------------------------------------------------------------------------- temperature matching (R6)
def test_temperature_matching(oracle_mod):
    from paper_1910_08448_b200 import inputs
    values, mask, truth = inputs.make_problem(64, 8.0, 0, 0.33)
    o = oracle_mod.Oracle(values=values, mask=mask, seed=1000)
    ladder = [1e-3, 1e-2, 3e-2, 1e-1, 3e-1, 1.0]
    es = [o.trial_energy(T, k + 1)[0] for k, T in enumerate(ladder)]
    assert all(b > a for a, b in zip(es, es[1:]))                       # e_cond(T) is monotone
    T_hat, e_s, n_trials = o.estimate_temperature()
    assert es[0] < e_s < es[-1]
    assert 2 <= n_trials <= 22
    # an independent seed at T_hat reproduces the sample energy
    o2 = oracle_mod.Oracle(values=values, mask=mask, seed=31337)
    o2.set_temperature(T_hat)
    _, e_mean, e_se = o2.run(300, 200)
    assert abs(e_mean - e_s) < 3.0 * math.hypot(e_se, 1e-4), (e_mean, e_s, e_se)
    # sanity bound of SURVEY 8c: the prediction beats the sample mean by a wide margin
    pred, _, _ = o.run(100, 100)
    mae, rmse = inputs.prediction_errors(pred, truth, mask)
    base = float(np.mean(np.abs(truth[mask == 1] - values[mask == 0].mean())))
    assert mae < 0.5 * base and rmse >= mae


def test_no_root_is_reported(oracle_mod):
    """Measured pairs perfectly aligned (e_s = -2) cannot be matched at any T > 0."""
    L = 12
    z = np.where(np.arange(L)[None, :] < 6, 10.0, 20.0) * np.ones((L, 1))
    rng = np.random.default_rng(0)
    mask = np.zeros((L, L), dtype=np.uint8)
    mask[:, 5:7] = 1                       # the step itself is hidden: every measured pair is equal
    mask[rng.integers(0, L, 20), rng.integers(0, 4, 20)] = 1
    vals = z.copy(); vals[mask == 1] = np.nan
    o = oracle_mod.Oracle(values=vals, mask=mask, seed=2)
    assert o.sample_energy()[0] == -2.0
    with pytest.raises(oracle_mod.OracleError) as ei:
        o.estimate_temperature()
    assert ei.value.code == oracle_mod.ERR_NO_ROOT


# --------------------------------------------------------------------------- general q (q in (0, 1/2])
@pytest.mark.parametrize("q", [0.5, 0.3, 0.1])
def test_general_q_energy_closed_forms(oracle_mod, q):
    """Uniform grid: e = -2J for every q.  I.i.d.-uniform spins: E cos[q(a - b)] = (E cos qa)^2 + (E sin qa)^2 =
    (2 - 2 cos 2 pi q) / (2 pi q)^2, so e -> -2J times that (4 / pi^2 at q = 1/2)."""
    L = 96
    o = oracle_mod.Oracle(phi=np.full((L, L), 1.234), mask=np.zeros((L, L), dtype=np.uint8))
    o.set_q(q)
    assert abs(o.energy()[1] + 2.0) <= 1e-12
    mask = np.ones((L, L), dtype=np.uint8)
    o = oracle_mod.Oracle(phi=np.zeros((L, L)), mask=mask)
    o.set_quench(0)
    o.set_q(q)
    o.set_seed(77)                                   # free spins i.i.d. uniform (R8 without the quench)
    expect = -2.0 * (2.0 - 2.0 * math.cos(TWO_PI * q)) / (TWO_PI * q) ** 2
    assert abs(o.energy()[1] - expect) < 5.0 / L     # ~ 1 / sqrt(number of bonds), generous


@pytest.mark.parametrize("q", [0.3, 0.1])
def test_general_q_over_relaxation(oracle_mod, q):
    """R5 at q < 1/2: the reflection phi' = 2 Phi / q - phi conserves H exactly and never leaves [0, 2 pi]
    (moves that would are dropped); applied twice it is the identity where it was accepted."""
    rng = np.random.default_rng(5)
    L = 24
    phi = rng.uniform(0.0, TWO_PI, (L, L))
    mask = (rng.uniform(size=(L, L)) < 0.8).astype(np.uint8)
    o = oracle_mod.Oracle(phi=phi, mask=mask)
    o.set_quench(0)
    o.set_q(q)
    o.set_state(phi)
    H0 = o.energy()[0]
    moved = 0
    for c in (0, 1, 0, 1):
        before = o.get_state()
        o.or_pass(c)
        after = o.get_state()
        moved += int((before != after).sum())
        assert abs(o.energy()[0] - H0) <= 1e-10 * abs(H0)
        assert after.min() >= 0.0 and after.max() <= TWO_PI
        assert np.array_equal(after[mask == 0], phi[mask == 0])
    assert moved > 0.1 * mask.sum()


@pytest.mark.parametrize("q,T", [(0.25, 0.1), (0.1, 0.02), (0.4, 1.0)])
def test_general_q_single_site_histogram(oracle_mod, q, T):
    """Hybrid sweeps at one free site with four fixed neighbours against p(phi) ~ exp(sum_j cos[q (phi - phi_j)] / T)."""
    (x, y), nbrs = SITE_CASES[0]
    L = 3
    phi = np.full((L, L), 3.0)
    for (a, b), v in nbrs.items():
        phi[b, a] = v
    mask = np.zeros((L, L), dtype=np.uint8)
    mask[y, x] = 1
    o = oracle_mod.Oracle(phi=phi, mask=mask)
    o.set_quench(0)
    o.set_q(q)
    o.set_seed(321)
    o.set_temperature(T)
    tr = o.trace(2_000_000, 1, [y * L + x])[1000::8, 0]
    xs = np.linspace(0.0, TWO_PI, 400001)
    logw = sum(np.cos(q * (xs - pj)) for pj in nbrs.values()) / T
    w = np.exp(logw - logw.max())
    cdf = np.concatenate([[0.0], np.cumsum(0.5 * (w[1:] + w[:-1]) * np.diff(xs))])
    cdf /= cdf[-1]
    nbins = 50
    edges = np.interp(np.linspace(0, 1, nbins + 1), cdf, xs)
    edges[0], edges[-1] = 0.0, TWO_PI
    counts, _ = np.histogram(tr, bins=edges)
    assert counts.sum() == tr.size
    chi2 = float(np.sum((counts - tr.size / nbins) ** 2 / (tr.size / nbins)))
    assert stats.chi2.sf(chi2, nbins - 1) > 1e-4, chi2


def test_general_q_proposal_width(oracle_mod):
    """delta = min(pi, 4 sqrt(T / (4 J q^2))) = min(pi, 2 sqrt(T) / q)."""
    assert oracle_mod.proposal_width(0.01, 0.25) == 0.8
    assert abs(oracle_mod.proposal_width(0.0025, 0.1) - 1.0) <= 1e-15
    assert oracle_mod.proposal_width(1.0, 0.1) == math.pi


# --------------------------------------------------------------------------- rectangular grids
def brute_force_H_rect(phi):
    """All pairs at Manhattan distance 1 on a (Ly, Lx) array -- no index arithmetic shared with the oracle."""
    Ly, Lx = phi.shape
    pts = [(x, y) for y in range(Ly) for x in range(Lx)]
    H = 0.0
    for i, (xa, ya) in enumerate(pts):
        for (xb, yb) in pts[i + 1:]:
            if abs(xa - xb) + abs(ya - yb) == 1:
                H -= math.cos(Q * (phi[ya, xa] - phi[yb, xb]))
    return H


@pytest.mark.parametrize("shape", [(3, 5), (5, 3), (1, 7), (7, 1), (2, 9), (6, 4)])
def test_rect_energy_vs_brute_force_and_transpose(oracle_mod, shape):
    """H on a rectangular grid = brute force over all unit-distance pairs; e = 2H / N_b with
    N_b = Lx (Ly - 1) + Ly (Lx - 1); the transposed field on the transposed grid has the same H (a row / column
    mix-up in the neighbour arithmetic breaks one of the three)."""
    Ly, Lx = shape
    rng = np.random.default_rng(100 * Ly + Lx)
    phi = rng.uniform(0, TWO_PI, (Ly, Lx))
    zero = np.zeros((Ly, Lx), dtype=np.uint8)
    o = oracle_mod.Oracle(phi=phi, mask=zero)
    H, e = o.energy()
    Hb = brute_force_H_rect(phi)
    nb = Lx * (Ly - 1) + Ly * (Lx - 1)
    assert abs(H - Hb) < 1e-12 * max(1.0, abs(Hb))
    assert abs(e - 2.0 * Hb / nb) < 1e-13
    ot = oracle_mod.Oracle(phi=np.ascontiguousarray(phi.T), mask=np.ascontiguousarray(zero.T))
    assert abs(ot.energy()[0] - H) < 1e-12 * max(1.0, abs(H))
    # aligned spins: every bond contributes -J, e = -2 whatever the shape
    oa = oracle_mod.Oracle(phi=np.full((Ly, Lx), 1.25), mask=zero)
    Ha, ea = oa.energy()
    assert abs(Ha + nb) < 1e-12 and abs(ea + 2.0) < 1e-14
    # local energy of every site = its part of H (sum over sites counts every bond twice)
    tot = sum(o.local_energy(x, y, phi[y, x]) for y in range(Ly) for x in range(Lx))
    assert abs(tot - 2.0 * Hb) < 1e-11


def test_rect_sample_energy_counts_measured_pairs_only(oracle_mod):
    Ly, Lx = 4, 7
    rng = np.random.default_rng(5)
    z = rng.uniform(0.0, TWO_PI, (Ly, Lx))
    mask = (rng.uniform(size=(Ly, Lx)) < 0.4).astype(np.uint8)
    mask[0, 0] = 0; mask[0, 1] = 0
    z[0, 0], z[0, 1] = 0.0, TWO_PI          # pins the range, so that phi = z
    z[mask == 1] = np.nan                    # never read
    o = oracle_mod.Oracle(values=z, mask=mask)
    es, n = o.sample_energy()
    s, cnt = 0.0, 0
    for y in range(Ly):
        for x in range(Lx):
            for (dx, dy) in ((1, 0), (0, 1)):
                xx, yy = x + dx, y + dy
                if xx < Lx and yy < Ly and not mask[y, x] and not mask[yy, xx]:
                    s += math.cos(Q * (z[y, x] - z[yy, xx])); cnt += 1
    assert n == cnt and abs(es + 2.0 * s / cnt) < 1e-13


RECT_SITE_CASES = [
    # (shape (Ly, Lx), free site (x, y), neighbour phis {(x, y): phi}) -- the free site has a DOWN neighbour in a row
    # index >= Lx (tall grid) or a RIGHT neighbour in a column index >= Ly (wide grid): a test of y against Lx or of
    # x against Ly drops it
    ((5, 2), (0, 3), {(1, 3): 0.7, (0, 2): 2.9, (0, 4): 5.1}),
    ((2, 6), (4, 1), {(3, 1): 1.3, (5, 1): 3.3, (4, 0): 0.2}),
    ((4, 3), (1, 2), {(0, 2): 1.0, (2, 2): 2.5, (1, 1): 4.0, (1, 3): 0.3}),
]


@pytest.mark.parametrize("schedule", ["R4", "SITE_FUSED"])
@pytest.mark.parametrize("case", [0, 1, 2], ids=["tall-edge3", "wide-edge3", "tall-interior4"])
def test_rect_single_site_histogram(oracle_mod, case, schedule):
    """The conditional density of one free site of a rectangular grid, hybrid sweeps, against the exact density."""
    (Ly, Lx), (x, y), nbrs = RECT_SITE_CASES[case]
    T = 0.1
    phi = np.full((Ly, Lx), 3.0)
    for (a, b), v in nbrs.items():
        phi[b, a] = v
    mask = np.zeros((Ly, Lx), dtype=np.uint8)
    mask[y, x] = 1
    o = oracle_mod.Oracle(phi=phi, mask=mask)
    o.set_quench(0)
    o.set_seed(4321 + case)
    o.set_temperature(T)
    o.set_schedule(schedule)
    thin = 8
    tr = o.trace(400_000 * thin // 4, 1, [y * Lx + x])[:, 0]
    chi2, p = chi2_against_density(tr[1000::thin], list(nbrs.values()), T)
    assert p > 1e-4, (chi2, p)
    st = o.get_state()
    for (a, b), v in nbrs.items():
        assert st[b, a] == v


def test_rect_chain_equals_square_chain_on_embedded_block(oracle_mod):
    """A rectangular problem is the same Markov chain as the square problem that contains it as a block walled off by
    measured sites -- but for the site indices the random numbers are keyed on.  What is index-free: a 1 x n chain
    of free sites between two measured ends at T -> 0 relaxes (quench passes) to the linear interpolation of the
    two end angles, the minimiser of sum cos[(phi_i - phi_i+1)/2], in a row and in a column alike."""
    n = 9
    for shape in ((1, n), (n, 1)):
        phi = np.zeros(shape); mask = np.ones(shape, dtype=np.uint8)
        flat_phi, flat_mask = phi.reshape(-1), mask.reshape(-1)
        flat_phi[0], flat_phi[-1] = 1.0, 3.0
        flat_mask[0] = flat_mask[-1] = 0
        o = oracle_mod.Oracle(phi=phi, mask=mask)
        o.set_seed(3)
        o.init_random(0)
        for _ in range(4000):
            o.quench_pass(0); o.quench_pass(1)
        st = o.get_state().reshape(-1)
        assert np.allclose(st, np.linspace(1.0, 3.0, n), atol=1e-6), st
