"""Host-side numerics, pinned on BOTH sides (the oracle's and the library's own, which share no text)
against things neither of them produced: hand-worked iterates, closed forms, and the root itself.

* R6, the temperature-matching root search (steps 1-5), on synthetic monotone
  e(T) handed in through orc_debug_match_temperature / mpr_debug_match_temperature.
* R16, the binned standard error, on series whose block statistics have closed forms.
* R7, the proposal half-width.

None of this needs a GPU: the library's hooks are host-only (include/mpr.h, "HOST-only hooks")."""
import math
from fractions import Fraction

import numpy as np
import pytest


@pytest.fixture(scope="module")
def sides(oracle_mod):
    from paper_1910_08448_b200 import build, mpr
    build.build()
    mpr.lib()

    def orc_match(es, f):
        st, T, asked = oracle_mod.match_temperature(es, f)
        return st, T, asked

    def lib_match(es, f):
        try:
            T, asked = mpr.debug_match_temperature(es, f)
            return 0, T, asked
        except mpr.MprError as err:
            return err.code, float("nan"), err.asked

    return {
        "oracle": dict(match=orc_match, stats=oracle_mod.mean_stderr, width=oracle_mod.proposal_width),
        "library": dict(match=lib_match, stats=mpr.debug_series_stats, width=mpr.debug_proposal_width),
    }


SIDES = ["oracle", "library"]


# ------------------------------------------------------------------------------------------ R6
@pytest.mark.parametrize("side", SIDES)
def test_illinois_iterates_worked_by_hand(sides, side):
    """e(T) = T^2, e_s = 1/4, standard error 0 (so only the |dT|/T < 1 % rule can stop it).  Root: T = 1/2.
    g(T) = T^2 - 1/4.  Worked by hand from R6 (6 significant digits):

      step 1   T = 1e-4            g = -0.25000        -> cold end
      step 3   T = 1               g = +0.75           -> warm end            bracket (1e-4, 1)
      step 4.1 T = 1 - 0.75 (1 - 1e-4)/(0.75 + 0.25)            = 0.250075    g = -0.187462  cold <- it
      step 4.2 T = 1 - 0.75 (1 - 0.250075)/(0.75 + 0.187462)    = 0.400036    g = -0.089971  cold <- it,
               the cold end was replaced twice running: the warm g is halved, 0.75 -> 0.375   (Illinois)
      step 4.3 T = 1 - 0.375 (1 - 0.400036)/(0.375 + 0.089971)  = 0.516128    g = +0.016388  warm <- it
      step 4.4 T = 0.516128 - 0.016388 (0.516128 - 0.400036)/(0.016388 + 0.089971) = 0.498240
               |0.498240 - 0.516128| / 0.498240 = 3.6 % >= 1 %: go on;          g = -0.001757  cold <- it
      step 4.5 T = 0.516128 - 0.016388 (0.516128 - 0.498240)/(0.016388 + 0.001757) = 0.499972
               |0.499972 - 0.498240| / 0.499972 = 0.35 % < 1 %: stop.  T_hat = 0.499972.

    Without the Illinois halving step 4.3 would be plain regula falsi, 1 - 0.75 (1 - 0.400036)/(0.75 +
    0.089971) = 0.464301: the test tells the two apart."""
    st, T, asked = sides[side]["match"](0.25, lambda T: (T * T, 0.0))
    assert st == 0
    hand = [1e-4, 1.0, 0.250075, 0.400036, 0.516128, 0.498240, 0.499972]
    assert len(asked) == len(hand), asked
    for a, h in zip(asked, hand):
        assert abs(a - h) <= 2e-6, (asked, hand)
    assert T == asked[-1]
    assert abs(T - 0.5) / 0.5 < 0.01                      # and it is the root, to the rule's own tolerance


def _r6_exact(e_of_T, e_s, se_of_T):
    """R6 steps 1-5 in exact rational arithmetic, written here from DESIGN.md's text."""
    asked = []

    def g(T):
        asked.append(T)
        return e_of_T(T) - e_s, se_of_T(T)

    a = Fraction(1, 10000)
    ga, _ = g(a)
    if ga > 0:
        while True:
            if a <= Fraction(15, 10 ** 7):
                return None, asked
            b, gb = a, ga
            a = a / 10
            ga, _ = g(a)
            if not ga > 0:
                break
    else:
        b = Fraction(1)
        gb, _ = g(b)
        while gb < 0:
            if b >= 99:
                return None, asked
            a, ga = b, gb
            b = b * 10
            gb, _ = g(b)
    last, prev, c = 0, None, b
    for it in range(20):
        c = b - gb * (b - a) / (gb - ga)
        if not (a < c < b):
            c = (a + b) / 2
        gc, sc = g(c)
        if abs(gc) <= 2 * sc:
            break
        if gc < 0:
            a, ga = c, gc
            if last == -1:
                gb = gb / 2
            last = -1
        else:
            b, gb = c, gc
            if last == +1:
                ga = ga / 2
            last = +1
        if it > 0 and abs(c - prev) / c < Fraction(1, 100):
            break
        prev = c
    return c, asked


CASES = [
    # (name, e(T) on Fractions, e_s, se(T))
    ("cubic, root 0.07", lambda T: T ** 3 + T, Fraction(7, 100) ** 3 + Fraction(7, 100), lambda T: Fraction(0)),
    ("concave, root 0.003", lambda T: T / (1 + T), Fraction(3, 1000) / (1 + Fraction(3, 1000)), lambda T: Fraction(0)),
    ("root below 1e-4: walk down by decades", lambda T: T * T, Fraction(3, 10 ** 5) ** 2, lambda T: Fraction(0)),
    ("root above 1: walk up by decades", lambda T: T, Fraction(37), lambda T: Fraction(0)),
    ("noise stop: |g| <= 2 se", lambda T: T, Fraction(1, 5), lambda T: Fraction(1, 20)),
]


@pytest.mark.parametrize("side", SIDES)
@pytest.mark.parametrize("name,e_of_T,e_s,se_of_T", CASES, ids=[c[0] for c in CASES])
def test_search_follows_r6_on_monotone_functions(sides, side, name, e_of_T, e_s, se_of_T):
    T_exact, asked_exact = _r6_exact(e_of_T, e_s, se_of_T)

    def f(T):
        Tf = Fraction(T)
        return float(e_of_T(Tf)), float(se_of_T(Tf))

    st, T, asked = sides[side]["match"](float(e_s), f)
    assert st == 0
    assert len(asked) == len(asked_exact), (asked, [float(t) for t in asked_exact])
    for a, b in zip(asked, asked_exact):
        assert abs(a - float(b)) <= 1e-9 * float(b), (asked, [float(t) for t in asked_exact])
    assert abs(T - float(T_exact)) <= 1e-9 * float(T_exact)
    if "noise" not in name:
        # the answer solves e(T) = e_s to the stop rule's 1 % (mathematics, not either implementation)
        lo, hi = 0.985 * T, 1.015 * T
        assert (e_of_T(Fraction(lo)) - e_s) * (e_of_T(Fraction(hi)) - e_s) < 0, name


@pytest.mark.parametrize("side", SIDES)
def test_no_root_cases(sides, side):
    # e(T) never comes down to e_s: decades 1e-4 ... 1e-6 are tried, then NO_ROOT (-7)
    st, _, asked = sides[side]["match"](-1.0, lambda T: (T, 0.0))
    assert st == -7
    np.testing.assert_allclose(asked, [1e-4, 1e-5, 1e-6], rtol=1e-12)
    # e(T) never reaches e_s: 1e-4, then 1, 10, 100, then NO_ROOT
    st, _, asked = sides[side]["match"](1e9, lambda T: (T, 0.0))
    assert st == -7
    np.testing.assert_allclose(asked, [1e-4, 1.0, 10.0, 100.0], rtol=1e-12)


@pytest.mark.parametrize("side", SIDES)
def test_search_is_bounded(sides, side):
    """A step function defeats the secant: at most 2 + 20 trials, and the answer sits at the step."""
    st, T, asked = sides[side]["match"](0.0, lambda T: (-1.0 if T < 0.3 else 5.0, 0.0))
    assert st == 0 and len(asked) <= 22
    assert abs(T - 0.3) / 0.3 < 0.02


# ------------------------------------------------------------------------------------------ R16
@pytest.mark.parametrize("side", SIDES)
def test_binned_standard_error_closed_forms(sides, side):
    stats = sides[side]["stats"]
    # 1..20: 10 blocks of 2 with means 1.5, 3.5, ..., 19.5 -- an arithmetic progression of step 2, whose
    # unbiased variance is step^2 B (B + 1) / 12 = 4 * 110 / 12; s.e. = sqrt(var / 10)
    m, s = stats(np.arange(1, 21, dtype=float))
    assert m == 10.5
    assert abs(s - math.sqrt(4 * 110 / 12 / 10)) <= 1e-14
    # 25 samples: block length floor(25 / 10) = 2, samples 21..25 enter the mean but no block
    m, s = stats(np.arange(1, 26, dtype=float))
    assert m == 13.0
    assert abs(s - math.sqrt(4 * 110 / 12 / 10)) <= 1e-14
    # fewer than 20 samples: every sample its own block -> the textbook standard error of the mean
    v = np.array([2.0, 4.0, 4.0, 4.0, 5.0, 5.0, 7.0, 9.0])      # mean 5, sum of squares 32
    m, s = stats(v)
    assert m == 5.0 and abs(s - math.sqrt(32 / 7 / 8)) <= 1e-15
    # a constant series has no error; one sample has none either; no sample: NaN mean
    assert stats(np.full(50, 3.25)) == (3.25, 0.0)
    assert stats(np.array([1.5])) == (1.5, 0.0)
    m, s = stats(np.array([]))
    assert math.isnan(m) and s == 0.0
    # blocks of 5: alternating +-1 inside a block cancel to +-1/5 -> block means (+0.2) x 10: s.e. 0
    v = np.tile([1.0, -1.0, 1.0, -1.0, 1.0], 10)
    m, s = stats(v)
    assert abs(m - 0.2) <= 1e-15 and s <= 1e-15


@pytest.mark.parametrize("side", SIDES)
def test_binned_standard_error_against_numpy(sides, side):
    rng = np.random.default_rng(5)
    for n in (2, 7, 19, 20, 50, 200, 203, 1000):
        v = rng.normal(-1.99, 1e-4, n)
        nb = 10 if n >= 20 else n
        ln = n // nb
        bm = v[:nb * ln].reshape(nb, ln).mean(axis=1)
        m, s = sides[side]["stats"](v)
        assert abs(m - math.fsum(v) / n) <= 2e-14          # naive summation of n terms near -2
        assert abs(s - math.sqrt(bm.var(ddof=1) / nb)) <= 1e-9 * s + 1e-16


# ------------------------------------------------------------------------------------------ R7
@pytest.mark.parametrize("side", SIDES)
def test_proposal_width(sides, side):
    """delta = min(pi, 4 sqrt(T / (4 J q^2))), q = 1/2, J = 1: delta = 4 sqrt(T) below the cap; the cap
    starts at T = (pi / 4)^2 = 0.61685."""
    w = sides[side]["width"]
    assert w(0.25) == 2.0
    assert w(1e-4) == 0.04
    assert abs(w(0.0011) - 4.0 * math.sqrt(0.0011)) <= 1e-16
    assert w(0.61) < math.pi and abs(w(0.61) - 4.0 * math.sqrt(0.61)) <= 1e-15
    assert w(0.62) == math.pi and w(1e6) == math.pi
    assert abs(w((math.pi / 4) ** 2) - math.pi) <= 1e-15
    # general q: delta = min(pi, 2 sqrt(T) / q)
    assert w(0.01, 0.25) == 0.8
    assert abs(w(0.0025, 0.1) - 1.0) <= 1e-15 and w(1.0, 0.1) == math.pi
