"""ctypes wrapper around oracle/mpr_oracle.cpp.

TEST INFRASTRUCTURE, NOT THE PRODUCT: only tests/, __graft_entry__.smoke() and bench.py's
cpu_baseline / --impl reference legs may import this module.  It imports nothing from the
CUDA package and the CUDA package imports nothing from here.
"""
from __future__ import annotations

import ctypes as C
import os
import subprocess

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "mpr_oracle.cpp")
_LIB = os.path.join(_HERE, "libmpr_oracle.so")

OK = 0
ERR_INVALID_ARG, ERR_NO_MEASURED, ERR_DEGENERATE_RANGE, ERR_NONFINITE = -1, -2, -3, -4
ERR_WORKSPACE, ERR_NOT_READY, ERR_NO_ROOT = -5, -6, -7


def build(force: bool = False) -> str:
    """Compile the oracle with gcc (no fused multiply-add contraction, OpenMP optional at run time)."""
    if force or not os.path.exists(_LIB) or os.path.getmtime(_LIB) < os.path.getmtime(_SRC):
        cmd = ["g++", "-O2", "-std=c++17", "-ffp-contract=off", "-fopenmp", "-shared", "-fPIC",
               "-Wall", "-Wextra", "-o", _LIB, _SRC]
        subprocess.run(cmd, check=True)
    return _LIB


TRIAL_FN = C.CFUNCTYPE(C.c_int, C.c_double, C.c_int, C.POINTER(C.c_double), C.POINTER(C.c_double), C.c_void_p)

_lib = None


def lib():
    global _lib
    if _lib is None:
        L = C.CDLL(build())
        dp, u8p, u32p, u64p, i64p = (C.POINTER(C.c_double), C.POINTER(C.c_uint8), C.POINTER(C.c_uint32),
                                     C.POINTER(C.c_uint64), C.POINTER(C.c_int64))
        vp = C.c_void_p
        sig = {
            "orc_philox4x32_10": (None, [u32p, u32p, u32p]),
            "orc_u53": (C.c_double, [C.c_uint32, C.c_uint32]),
            "orc_proposal_width": (C.c_double, [C.c_double]),
            "orc_mean_stderr": (None, [dp, C.c_long, dp, dp]),
            "orc_create": (vp, [C.c_int, dp, u8p, C.POINTER(C.c_int)]),
            "orc_create_deferred": (vp, [C.c_int, dp, u8p, C.POINTER(C.c_int)]),
            "orc_configure": (C.c_int, [vp, C.c_uint64, C.c_int]),
            "orc_create_from_phi": (vp, [C.c_int, dp, u8p]),
            "orc_create_rect": (vp, [C.c_int, C.c_int, dp, u8p, C.POINTER(C.c_int)]),
            "orc_create_rect_deferred": (vp, [C.c_int, C.c_int, dp, u8p, C.POINTER(C.c_int)]),
            "orc_create_from_phi_rect": (vp, [C.c_int, C.c_int, dp, u8p]),
            "orc_destroy": (None, [vp]),
            "orc_set_seed": (C.c_int, [vp, C.c_uint64]),
            "orc_set_temperature": (C.c_int, [vp, C.c_double]),
            "orc_set_quench": (C.c_int, [vp, C.c_int]),
            "orc_set_threads": (C.c_int, [vp, C.c_int]),
            "orc_set_schedule": (C.c_int, [vp, C.c_int]),
            "orc_set_q": (C.c_int, [vp, C.c_double]),
            "orc_proposal_width_q": (C.c_double, [C.c_double, C.c_double]),
            "orc_threads_available": (C.c_int, []),
            "orc_reset_chain": (None, [vp, C.c_uint32]),
            "orc_init_random": (None, [vp, C.c_uint32]),
            "orc_get_range": (None, [vp, dp, dp]),
            "orc_met_pass": (C.c_int, [vp, C.c_int, C.c_uint64]),
            "orc_or_pass": (None, [vp, C.c_int]),
            "orc_quench_pass": (None, [vp, C.c_int]),
            "orc_hybrid_sweeps": (C.c_int, [vp, C.c_int]),
            "orc_trace": (C.c_int, [vp, C.c_long, C.c_int, i64p, C.c_int, dp]),
            "orc_trace_energy": (C.c_int, [vp, C.c_long, dp]),
            "orc_energy": (None, [vp, dp, dp]),
            "orc_sample_energy": (C.c_int, [vp, dp, C.POINTER(C.c_longlong)]),
            "orc_local_energy": (C.c_double, [vp, C.c_int, C.c_int, C.c_double]),
            "orc_get_state": (None, [vp, dp]),
            "orc_set_state": (None, [vp, dp]),
            "orc_get_counters": (None, [vp, u64p, u64p, u64p]),
            "orc_run": (C.c_int, [vp, C.c_int, C.c_int, dp, dp, dp]),
            "orc_get_series": (C.c_long, [vp, dp, C.c_long]),
            "orc_estimate_temperature": (C.c_int, [vp, dp, dp, C.POINTER(C.c_int)]),
            "orc_trial_energy": (C.c_int, [vp, C.c_double, C.c_int, dp, dp]),
            "orc_debug_match_temperature": (C.c_int, [C.c_double, TRIAL_FN, vp, dp, C.POINTER(C.c_int)]),
        }
        for name, (res, args) in sig.items():
            fn = getattr(L, name)
            fn.restype, fn.argtypes = res, args
        _lib = L
    return _lib


def _dp(a):
    return a.ctypes.data_as(C.POINTER(C.c_double))


class OracleError(RuntimeError):
    def __init__(self, code):
        super().__init__(f"oracle status {code}")
        self.code = code


def philox4x32_10(ctr, key):
    c = (C.c_uint32 * 4)(*[int(v) & 0xFFFFFFFF for v in ctr])
    k = (C.c_uint32 * 2)(*[int(v) & 0xFFFFFFFF for v in key])
    o = (C.c_uint32 * 4)()
    lib().orc_philox4x32_10(c, k, o)
    return [int(v) for v in o]


def u53(a, b):
    return lib().orc_u53(int(a), int(b))


def proposal_width(T, q=None):
    return lib().orc_proposal_width(float(T)) if q is None else lib().orc_proposal_width_q(float(T), float(q))


def mean_stderr(v):
    v = np.ascontiguousarray(v, dtype=np.float64)
    m, s = C.c_double(), C.c_double()
    lib().orc_mean_stderr(_dp(v), len(v), C.byref(m), C.byref(s))
    return m.value, s.value


class Oracle:
    """One MPR problem held by the CPU oracle.  `mask` = 1 marks a prediction site."""

    def __init__(self, values=None, mask=None, phi=None, seed=None, threads=1, n_quench=None):
        """n_quench given: large-grid form -- the chain is initialised once, on `threads` threads, with
        (seed, n_quench) (orc_create_deferred + orc_configure) instead of once per setter."""
        L_ = lib()
        mask = np.ascontiguousarray(mask, dtype=np.uint8)
        # mask.shape = (Ly rows, Lx columns); L is kept as the name of the size of a square grid
        self.Ly, self.Lx = int(mask.shape[0]), int(mask.shape[1])
        self.L = self.Ly if self.Ly == self.Lx else None
        self.shape = (self.Ly, self.Lx)
        self.mask = mask
        if phi is not None:
            phi = np.ascontiguousarray(phi, dtype=np.float64)
            assert phi.shape == self.shape
            self.h = L_.orc_create_from_phi_rect(self.Lx, self.Ly, _dp(phi), mask.ctypes.data_as(C.POINTER(C.c_uint8)))
            if not self.h:
                raise OracleError(ERR_INVALID_ARG)
        else:
            values = np.ascontiguousarray(values, dtype=np.float64)
            st = C.c_int()
            assert values.shape == self.shape
            create = L_.orc_create_rect if n_quench is None else L_.orc_create_rect_deferred
            self.h = create(self.Lx, self.Ly, _dp(values), mask.ctypes.data_as(C.POINTER(C.c_uint8)), C.byref(st))
            if not self.h:
                raise OracleError(st.value)
            if n_quench is not None:
                self.set_threads(threads)
                self._chk(L_.orc_configure(self.h, int(seed or 0), int(n_quench)))
                return
        if threads != 1:
            self.set_threads(threads)
        if seed is not None:
            self.set_seed(seed)

    def __del__(self):
        h = getattr(self, "h", None)
        if h:
            lib().orc_destroy(h)
            self.h = None

    def _chk(self, st):
        if st != OK:
            raise OracleError(st)

    def set_seed(self, seed):
        self._chk(lib().orc_set_seed(self.h, int(seed)))

    def set_temperature(self, T):
        self._chk(lib().orc_set_temperature(self.h, float(T)))

    def set_quench(self, n):
        self._chk(lib().orc_set_quench(self.h, int(n)))

    def set_q(self, q):
        self._chk(lib().orc_set_q(self.h, float(q)))

    def set_schedule(self, schedule):
        """"R4" (default) or "SITE_FUSED" (R4b): the order of the four colour passes of a hybrid sweep."""
        self._chk(lib().orc_set_schedule(self.h, {"R4": 0, "SITE_FUSED": 1}[schedule]))

    def set_threads(self, n):
        self._chk(lib().orc_set_threads(self.h, int(n)))

    def reset_chain(self, trial=0):
        lib().orc_reset_chain(self.h, int(trial))

    def init_random(self, trial=0):
        lib().orc_init_random(self.h, int(trial))

    def zrange(self):
        a, b = C.c_double(), C.c_double()
        lib().orc_get_range(self.h, C.byref(a), C.byref(b))
        return a.value, b.value

    def met_pass(self, c, n):
        self._chk(lib().orc_met_pass(self.h, int(c), int(n)))

    def or_pass(self, c):
        lib().orc_or_pass(self.h, int(c))

    def quench_pass(self, c):
        lib().orc_quench_pass(self.h, int(c))

    def hybrid_sweeps(self, n=1):
        self._chk(lib().orc_hybrid_sweeps(self.h, int(n)))

    def trace(self, n, kind, sites):
        sites = np.ascontiguousarray(sites, dtype=np.int64)
        out = np.empty((int(n), len(sites)), dtype=np.float64)
        self._chk(lib().orc_trace(self.h, int(n), int(kind), sites.ctypes.data_as(C.POINTER(C.c_int64)),
                                  len(sites), _dp(out)))
        return out

    def trace_energy(self, n):
        out = np.empty(int(n), dtype=np.float64)
        self._chk(lib().orc_trace_energy(self.h, int(n), _dp(out)))
        return out

    def energy(self):
        H, e = C.c_double(), C.c_double()
        lib().orc_energy(self.h, C.byref(H), C.byref(e))
        return H.value, e.value

    def sample_energy(self):
        es, n = C.c_double(), C.c_longlong()
        self._chk(lib().orc_sample_energy(self.h, C.byref(es), C.byref(n)))
        return es.value, n.value

    def local_energy(self, x, y, phi_s):
        return lib().orc_local_energy(self.h, int(x), int(y), float(phi_s))

    def get_state(self):
        out = np.empty(self.shape, dtype=np.float64)
        lib().orc_get_state(self.h, _dp(out))
        return out

    def set_state(self, phi):
        phi = np.ascontiguousarray(phi, dtype=np.float64)
        assert phi.shape == self.shape
        lib().orc_set_state(self.h, _dp(phi))

    def counters(self):
        a, b, c = C.c_uint64(), C.c_uint64(), C.c_uint64()
        lib().orc_get_counters(self.h, C.byref(a), C.byref(b), C.byref(c))
        return a.value, b.value, c.value

    def run(self, n_eq, n_meas):
        pred = np.empty(self.shape, dtype=np.float64)
        m, s = C.c_double(), C.c_double()
        self._chk(lib().orc_run(self.h, int(n_eq), int(n_meas), _dp(pred), C.byref(m), C.byref(s)))
        return pred, m.value, s.value

    def series(self):
        n = lib().orc_get_series(self.h, None, 0)
        out = np.empty(n, dtype=np.float64)
        lib().orc_get_series(self.h, _dp(out), n)
        return out

    def estimate_temperature(self):
        T, es, nt = C.c_double(), C.c_double(), C.c_int()
        self._chk(lib().orc_estimate_temperature(self.h, C.byref(T), C.byref(es), C.byref(nt)))
        return T.value, es.value, nt.value

    def trial_energy(self, T, trial_index=1):
        e, se = C.c_double(), C.c_double()
        self._chk(lib().orc_trial_energy(self.h, float(T), int(trial_index), C.byref(e), C.byref(se)))
        return e.value, se.value


def match_temperature(e_sample, energy_of_T):
    """The oracle's R6 search on a Python function T -> (e, se).  Returns (status, T_hat, [T asked])."""
    asked = []

    def cb(T, idx, e, se, _user):
        asked.append(T)
        e[0], se[0] = energy_of_T(T)
        return 0

    T, n = C.c_double(), C.c_int()
    st = lib().orc_debug_match_temperature(float(e_sample), TRIAL_FN(cb), None, C.byref(T), C.byref(n))
    return st, T.value, asked


def threads_available():
    return lib().orc_threads_available()
