"""Seeded synthetic inputs with the structure of the paper's workload (Eq. 3).

The paper's fields are Gaussian N(50, 10) with exponential covariance sigma^2 exp(-kappa h)
on L x L grids with a share of the points removed uniformly at random.  Its realisations are
not available; BASELINE.json's `configs` stand in with the same family: Whittle-Matern nu = 0.5
(the exponential covariance, xi = 1/kappa) by FFT spectral synthesis, plus one lognormal field.

This module serves both the CPU oracle's tests and the CUDA path's tests / bench.  It holds
none of the method's arithmetic and imports neither of them; numpy / scipy only.
"""
from __future__ import annotations

import hashlib
from dataclasses import dataclass

import numpy as np

try:  # multi-threaded pocketfft; same algorithm family as numpy.fft
    import scipy.fft as _fft
    _FFT_KW = {"workers": -1}
except Exception:  # pragma: no cover
    import numpy.fft as _fft
    _FFT_KW = {}


@dataclass(frozen=True)
class Config:
    name: str
    L: int
    xi: float
    field_seed: int
    f: float
    lognormal: bool
    mpr_seed: int
    n_eq: int
    n_meas: int
    modes: tuple


# BASELINE.json `configs`, in order.  Modes use the C-ABI enum names.
CONFIGS = {
    1: Config("config1_L64", 64, 8.0, 0, 0.33, False, 1000, 100, 100, ("DP",)),
    2: Config("config2_L512", 512, 32.0, 1, 0.66, False, 1001, 1000, 100, ("DP", "SP")),
    3: Config("config3_L2048_lognormal", 2048, 64.0, 2, 0.33, True, 1002, 1000, 100,
              ("DP", "SP", "SP_PRECISE", "SP_INTRINSIC")),
    4: Config("config4_L8192", 8192, 128.0, 3, 0.66, False, 1003, 2000, 200, ("SP", "SP_INTRINSIC")),
    5: Config("config5_L16384", 16384, 256.0, 4, 0.90, False, 1004, 2000, 200,
              ("DP", "SP", "SP_PRECISE", "SP_INTRINSIC")),
}


def matern_field(L: int, xi: float, rng: np.random.Generator, nu: float = 0.5) -> np.ndarray:
    """Unit-variance periodic Gaussian random field with the 2-D Matern spectrum (xi^-2 + k^2)^-(nu+1)."""
    W = rng.standard_normal((L, L))
    kx = 2.0 * np.pi * np.fft.fftfreq(L)
    ky = 2.0 * np.pi * np.fft.rfftfreq(L)
    F = _fft.rfft2(W, **_FFT_KW)
    del W
    S = (xi ** -2 + kx[:, None] ** 2 + ky[None, :] ** 2) ** (-(nu + 1.0))
    np.sqrt(S, out=S)
    F *= S
    del S
    g = _fft.irfft2(F, s=(L, L), **_FFT_KW)
    del F
    g -= g.mean()
    g /= g.std()
    return g


def make_problem(L: int, xi: float, field_seed: int, f: float, lognormal: bool = False,
                 mean: float = 50.0, std: float = 10.0):
    """Returns (values, mask, truth): float64[L,L] with NaN at prediction sites, uint8[L,L]
    (1 = prediction site), float64[L,L] complete field."""
    rng = np.random.default_rng(field_seed)
    g = matern_field(L, xi, rng)
    if lognormal:
        z = np.exp(g)
    else:
        z = mean + std * g
    del g
    n_pred = int(round(f * L * L))
    idx = rng.choice(L * L, size=n_pred, replace=False, shuffle=False)
    mask = np.zeros(L * L, dtype=np.uint8)
    mask[idx] = 1
    del idx
    mask = mask.reshape(L, L)
    truth = z
    values = z.copy()
    values[mask == 1] = np.nan
    return values, mask, truth


def make_rect_problem(Ly: int, Lx: int, xi: float, field_seed: int, f: float, lognormal: bool = False):
    """A rectangular problem (Ly rows, Lx columns): the top-left Ly x Lx window of the square problem of
    side max(Ly, Lx), with its mask (the masked fraction of the window is close to f, not exactly f).  A window that
    came out with fewer than two measured sites gets its first two sites measured."""
    values, mask, truth = make_problem(max(Ly, Lx), xi, field_seed, f, lognormal)
    values = np.ascontiguousarray(values[:Ly, :Lx]); mask = np.ascontiguousarray(mask[:Ly, :Lx])
    truth = np.ascontiguousarray(truth[:Ly, :Lx])
    if int((mask == 0).sum()) < 2:
        flat_m, flat_v, flat_t = mask.reshape(-1), values.reshape(-1), truth.reshape(-1)
        flat_m[:2] = 0
        flat_v[:2] = flat_t[:2]
    return values, mask, truth


def structured_mask(L: int, kind: str, f: float, seed: int) -> np.ndarray:
    """Gap patterns of remote-sensing data ("restricted satellite paths or bad weather conditions"),
    uint8[L, L] with 1 = prediction site and a masked fraction close to f:
      "clouds"  -- the sites where a smooth Gaussian random field (correlation length L / 16) exceeds its (1 - f) quantile:
                   compact blobs with ragged edges;
      "tracks"  -- everything EXCEPT diagonal swaths (the satellite paths) of equal width, one every L / 8 columns, whose
                   width is set so that the swaths cover 1 - f of the grid."""
    rng = np.random.default_rng(seed)
    if kind == "clouds":
        g = matern_field(L, max(2.0, L / 16.0), rng, nu=1.5)
        thr = np.quantile(g, 1.0 - f)
        return (g > thr).astype(np.uint8)
    if kind == "tracks":
        period = max(8, L // 8)
        width = max(1, int(round((1.0 - f) * period)))
        y, x = np.mgrid[0:L, 0:L]
        phase = int(rng.integers(0, period))
        seen = ((x + (y // 3) + phase) % period) < width          # swaths inclined by 1 : 3
        return (~seen).astype(np.uint8)
    raise ValueError(kind)


def make_structured_problem(L: int, xi: float, field_seed: int, f: float, kind: str):
    """make_problem with a structured gap pattern instead of uniformly scattered prediction sites."""
    rng = np.random.default_rng(field_seed)
    z = 50.0 + 10.0 * matern_field(L, xi, rng)
    mask = structured_mask(L, kind, f, field_seed + 7919)
    values = z.copy()
    values[mask == 1] = np.nan
    return values, mask, z


def make_config(i: int):
    c = CONFIGS[i]
    return (c,) + make_problem(c.L, c.xi, c.field_seed, c.f, c.lognormal)


def sha256(a: np.ndarray) -> str:
    return hashlib.sha256(np.ascontiguousarray(a).tobytes()).hexdigest()


def prediction_errors(pred: np.ndarray, truth: np.ndarray, mask: np.ndarray):
    """MAE (the paper's AAE, Eq. 4) and RMSE over the prediction sites."""
    m = mask.astype(bool)
    d = pred[m] - truth[m]
    return float(np.mean(np.abs(d))), float(np.sqrt(np.mean(d * d)))
