"""Thin ctypes binding of libmpr.so (include/mpr.h): argument marshalling only.

Every step of the path runs in the CUDA kernels of the library; torch is used for device
memory and streams.  There is no CPU fallback: importing works without a GPU (so that the
symbol table can be checked), every compute call needs one and fails loudly otherwise.
"""
from __future__ import annotations

import ctypes as C
import os

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(_HERE, "libmpr.so")

MPR_OK = 0
ERR_INVALID_ARG, ERR_NO_MEASURED, ERR_DEGENERATE_RANGE, ERR_NONFINITE = -1, -2, -3, -4
ERR_WORKSPACE, ERR_NOT_READY, ERR_NO_ROOT, ERR_CUDA = -5, -6, -7, -8

MODES = {"DP": 0, "SP": 1, "SP_PRECISE": 2, "SP_INTRINSIC": 3, "DS_INTRINSIC": 4, "HP": 5}
TRIPLES = ("DDD", "DSD", "DDS", "SDD", "SDS", "DSS", "SSD", "SSS")      # PAPER.md:35, in Fig. 2's order after DDD
PATHS = {"TILED": 0, "PLAIN": 1, "STRIP": 2, "AUTO": 3, "LIST": 4}
SCHEDULES = {"R4": 0, "SITE_FUSED": 1}
PASS_KINDS = {"MET": 0, "OR": 1, "QUENCH": 2, "MO": 3}

# every symbol include/mpr.h declares
SYMBOLS = [
    "mpr_workspace_bytes", "mpr_create", "mpr_destroy", "mpr_set_workspace", "mpr_set_stream",
    "mpr_debug_series_stats", "mpr_debug_match_temperature", "mpr_debug_proposal_width", "mpr_set_precision",
    "mpr_set_precision_triple", "mpr_set_energy_precision", "mpr_set_q", "mpr_debug_proposal_width_q", "mpr_set_seed",
    "mpr_set_temperature", "mpr_set_quench", "mpr_set_path", "mpr_set_fused_sweeps", "mpr_set_schedule", "mpr_reset_chain",
    "mpr_estimate_temperature", "mpr_run", "mpr_sweep", "mpr_pass", "mpr_get_state", "mpr_set_state",
    "mpr_energy", "mpr_sample_energy", "mpr_get_counters", "mpr_get_run_timing", "mpr_get_energy_series",
    "mpr_get_info",
    "mpr_get_launch_stats", "mpr_workspace_bytes_host", "mpr_predict_host", "mpr_debug_philox",
    "mpr_workspace_bytes_rect", "mpr_create_rect", "mpr_workspace_bytes_host_rect", "mpr_predict_host_rect",
    "mpr_create_slab", "mpr_set_slab", "mpr_set_peers", "mpr_sample_energy_parts", "mpr_rows_bytes", "mpr_export_rows", "mpr_import_rows", "mpr_advance",
    "mpr_fetch_series", "mpr_predict", "mpr_debug_trial_lengths", "mpr_quench",
    "mpr_debug_accept",
    "mpr_static_setup", "mpr_static_max_sites", "mpr_static_last_error", "mpr_sample_energy_static",
    "mpr_last_error", "mpr_status_string",
]

# int trial(double T, int trial_index, double* e, double* se, void* user) -- mpr_debug_match_temperature
TRIAL_FN = C.CFUNCTYPE(C.c_int, C.c_double, C.c_int, C.POINTER(C.c_double), C.POINTER(C.c_double), C.c_void_p)

_lib = None


class MprError(RuntimeError):
    def __init__(self, code, msg=""):
        super().__init__("libmpr status %d (%s) %s" % (code, _status_string(code), msg))
        self.code = code


def _status_string(code):
    try:
        return lib().mpr_status_string(int(code)).decode()
    except Exception:
        return "?"


def lib():
    """Loads libmpr.so (building it first if the sources are newer).  Raises if it is missing."""
    global _lib
    if _lib is not None:
        return _lib
    if not os.path.exists(LIB_PATH):
        from . import build as _build
        _build.build()
    L = C.CDLL(LIB_PATH)
    vp, dp, i64 = C.c_void_p, C.POINTER(C.c_double), C.c_int64
    u64p, i64p = C.POINTER(C.c_uint64), C.POINTER(C.c_int64)
    sig = {
        "mpr_workspace_bytes": (C.c_int, [C.c_int, C.POINTER(C.c_size_t)]),
        "mpr_create": (C.c_int, [C.POINTER(vp), C.c_int, vp, vp, vp, C.c_size_t, vp]),
        "mpr_workspace_bytes_rect": (C.c_int, [C.c_int, C.c_int, C.POINTER(C.c_size_t)]),
        "mpr_create_rect": (C.c_int, [C.POINTER(vp), C.c_int, C.c_int, vp, vp, vp, C.c_size_t, vp]),
        "mpr_workspace_bytes_host_rect": (C.c_int, [C.c_int, C.c_int, C.POINTER(C.c_size_t)]),
        "mpr_predict_host_rect": (C.c_int, [C.c_int, C.c_int, vp, vp, C.c_int, C.c_uint64, C.c_double, C.c_int, C.c_int,
                                            vp, C.c_size_t, vp, vp, dp, dp, dp, u64p]),
        "mpr_destroy": (None, [vp]),
        "mpr_set_workspace": (C.c_int, [vp, vp, C.c_size_t]),
        "mpr_set_stream": (C.c_int, [vp, vp]),
        "mpr_debug_proposal_width": (C.c_double, [C.c_double]),
        "mpr_debug_series_stats": (C.c_int, [dp, i64, dp, dp]),
        "mpr_debug_match_temperature": (C.c_int, [C.c_double, TRIAL_FN, vp, dp, C.POINTER(C.c_int)]),
        "mpr_set_precision": (C.c_int, [vp, C.c_int]),
        "mpr_set_precision_triple": (C.c_int, [vp, C.c_char_p]),
        "mpr_set_energy_precision": (C.c_int, [vp, C.c_int]),
        "mpr_set_q": (C.c_int, [vp, C.c_double]),
        "mpr_debug_proposal_width_q": (C.c_double, [C.c_double, C.c_double]),
        "mpr_set_seed": (C.c_int, [vp, C.c_uint64]),
        "mpr_set_temperature": (C.c_int, [vp, C.c_double]),
        "mpr_set_quench": (C.c_int, [vp, C.c_int]),
        "mpr_set_path": (C.c_int, [vp, C.c_int]),
        "mpr_set_fused_sweeps": (C.c_int, [vp, C.c_int]),
        "mpr_set_schedule": (C.c_int, [vp, C.c_int]),
        "mpr_reset_chain": (C.c_int, [vp, C.c_uint32]),
        "mpr_estimate_temperature": (C.c_int, [vp, dp, dp, C.POINTER(C.c_int)]),
        "mpr_run": (C.c_int, [vp, C.c_int, C.c_int, vp, dp, dp]),
        "mpr_sweep": (C.c_int, [vp, C.c_int]),
        "mpr_pass": (C.c_int, [vp, C.c_int, C.c_int, C.c_uint64]),
        "mpr_get_state": (C.c_int, [vp, vp]),
        "mpr_set_state": (C.c_int, [vp, vp]),
        "mpr_energy": (C.c_int, [vp, dp, dp]),
        "mpr_sample_energy": (C.c_int, [vp, dp, i64p]),
        "mpr_get_counters": (C.c_int, [vp, u64p, u64p, u64p]),
        "mpr_get_run_timing": (C.c_int, [vp, dp, i64p, i64p]),
        "mpr_get_energy_series": (i64, [vp, dp, i64]),
        "mpr_get_info": (C.c_int, [vp, dp, dp, i64p, dp]),
        "mpr_get_launch_stats": (C.c_int, [vp, u64p]),
        "mpr_workspace_bytes_host": (C.c_int, [C.c_int, C.POINTER(C.c_size_t)]),
        "mpr_predict_host": (C.c_int, [C.c_int, vp, vp, C.c_int, C.c_uint64, C.c_double, C.c_int, C.c_int, vp,
                                       C.c_size_t, vp, vp, dp, dp, dp, u64p]),
        "mpr_debug_philox": (C.c_int, [vp, C.POINTER(C.c_uint32), vp, i64, vp]),
        "mpr_create_slab": (C.c_int, [C.POINTER(vp), C.c_int, C.c_int, vp, vp, vp, C.c_size_t, vp]),
        "mpr_set_slab": (C.c_int, [vp, C.c_int, C.c_int, C.c_int, C.c_double, C.c_double, C.c_double]),
        "mpr_sample_energy_parts": (C.c_int, [vp, dp, i64p]),
        "mpr_set_peers": (C.c_int, [vp, vp, vp]),
        "mpr_rows_bytes": (C.c_int, [vp, C.c_int, C.POINTER(C.c_size_t)]),
        "mpr_export_rows": (C.c_int, [vp, C.c_int, C.c_int, vp]),
        "mpr_import_rows": (C.c_int, [vp, C.c_int, C.c_int, vp]),
        "mpr_advance": (C.c_int, [vp, C.c_int, C.c_int, C.c_int]),
        "mpr_fetch_series": (C.c_int, [vp, C.c_int, dp]),
        "mpr_quench": (C.c_int, [vp, C.c_int]),
        "mpr_predict": (C.c_int, [vp, vp]),
        "mpr_debug_trial_lengths": (None, [C.POINTER(C.c_int), C.POINTER(C.c_int)]),
        "mpr_debug_accept": (C.c_int, [vp, vp, C.c_double, vp, i64, vp]),
        "mpr_static_setup": (C.c_int, []),
        "mpr_static_max_sites": (C.c_int64, []),
        "mpr_static_last_error": (C.c_char_p, []),
        "mpr_sample_energy_static": (C.c_int, [C.c_int, C.c_int, vp, vp, C.c_double, vp, vp]),
        "mpr_last_error": (C.c_char_p, [vp]),
        "mpr_status_string": (C.c_char_p, [C.c_int]),
    }
    for name, (res, args) in sig.items():
        fn = getattr(L, name)
        fn.restype, fn.argtypes = res, args
    _lib = L
    return L


def workspace_bytes(L, host: bool = False) -> int:
    """L: the size of a square grid, or a shape (Ly rows, Lx columns)."""
    n = C.c_size_t()
    if isinstance(L, (tuple, list)):
        fn = lib().mpr_workspace_bytes_host_rect if host else lib().mpr_workspace_bytes_rect
        st = fn(int(L[1]), int(L[0]), C.byref(n))
    else:
        fn = lib().mpr_workspace_bytes_host if host else lib().mpr_workspace_bytes
        st = fn(int(L), C.byref(n))
    if st != MPR_OK:
        raise MprError(st)
    return n.value


def _torch():
    import torch
    if not torch.cuda.is_available():
        raise RuntimeError("paper_1910_08448_b200 needs a CUDA device: there is no CPU fallback")
    return torch


class Mpr:
    """One MPR prediction problem on the GPU.  Mirrors the C calls of include/mpr.h by name.

    values: float64 [L, L] (torch CUDA tensor or numpy array; NaN allowed at prediction sites)
    mask:   uint8   [L, L], 1 = prediction site
    """

    def __init__(self, values, mask, mode="DP", seed=None, device="cuda:0", stream=None, slab=False):
        torch = _torch()
        self._torch = torch
        dev = torch.device(device)
        self.values = torch.as_tensor(values, dtype=torch.float64).to(dev).contiguous()
        self.mask = torch.as_tensor(mask, dtype=torch.uint8).to(dev).contiguous()
        # shape = (Ly rows, Lx columns); L names the size of a square grid (None otherwise)
        self.Ly, self.Lx = int(self.mask.shape[0]), int(self.mask.shape[1])
        self.shape = (self.Ly, self.Lx)
        self.L = self.Ly if self.Ly == self.Lx else None
        assert self.mask.dim() == 2 and tuple(self.values.shape) == self.shape
        self.device = dev
        self.ws = torch.empty(workspace_bytes(self.shape) + 256, dtype=torch.uint8, device=dev)
        off = (-self.ws.data_ptr()) % 256
        self._ws_ptr = self.ws.data_ptr() + off
        self._stream = stream
        sptr = stream.cuda_stream if stream is not None else torch.cuda.current_stream(dev).cuda_stream
        self.h = C.c_void_p()
        # bound here so that close() works from __del__ at interpreter shutdown, when module
        # globals (lib, C) may already be cleared
        self._destroy, self._null = lib().mpr_destroy, C.c_void_p
        with torch.cuda.device(dev):
            if slab:        # rows that will become a slab (mpr_create_slab): set_slab must follow
                st = lib().mpr_create_slab(C.byref(self.h), self.Lx, self.Ly, self.values.data_ptr(), self.mask.data_ptr(),
                                           self._ws_ptr, self.ws.numel() - off, sptr)
            elif self.L is not None:
                st = lib().mpr_create(C.byref(self.h), self.L, self.values.data_ptr(), self.mask.data_ptr(),
                                      self._ws_ptr, self.ws.numel() - off, sptr)
            else:
                st = lib().mpr_create_rect(C.byref(self.h), self.Lx, self.Ly, self.values.data_ptr(), self.mask.data_ptr(),
                                           self._ws_ptr, self.ws.numel() - off, sptr)
        if st != MPR_OK:
            self.h = C.c_void_p()
            raise MprError(st)
        if mode != "DP":
            self.set_precision(mode)
        if seed is not None:
            self.set_seed(seed)

    def close(self):
        h = getattr(self, "h", None)
        if h is not None and h.value and getattr(self, "_destroy", None) is not None:
            self._destroy(h)
            self.h = self._null()

    __del__ = close

    def _chk(self, st):
        if st != MPR_OK:
            raise MprError(st, lib().mpr_last_error(self.h).decode())

    def _call(self, fn, *args):
        with self._torch.cuda.device(self.device):
            self._chk(fn(self.h, *args))

    # -- setters -------------------------------------------------------------------------
    def set_workspace(self, ws):
        """Attach another caller-owned workspace tensor (uint8, CUDA)."""
        off = (-ws.data_ptr()) % 256
        self._call(lib().mpr_set_workspace, ws.data_ptr() + off, ws.numel() - off)
        self.ws = ws

    def set_stream(self, stream):
        self._call(lib().mpr_set_stream, stream.cuda_stream if stream is not None else None)
        self._stream = stream

    def set_precision(self, mode):
        self._call(lib().mpr_set_precision, MODES[mode] if isinstance(mode, str) else int(mode))

    def set_precision_triple(self, triple):
        self._call(lib().mpr_set_precision_triple, triple.encode())

    def set_q(self, q):
        self._call(lib().mpr_set_q, float(q))

    def set_energy_precision(self, single):
        self._call(lib().mpr_set_energy_precision, 1 if single else 0)

    def set_seed(self, seed):
        self._call(lib().mpr_set_seed, int(seed))

    def set_temperature(self, T):
        self._call(lib().mpr_set_temperature, float(T))

    def set_quench(self, n):
        self._call(lib().mpr_set_quench, int(n))

    def set_path(self, path):
        self._call(lib().mpr_set_path, PATHS[path] if isinstance(path, str) else int(path))

    def set_schedule(self, schedule):
        self._call(lib().mpr_set_schedule, SCHEDULES[schedule] if isinstance(schedule, str) else int(schedule))

    def set_fused_sweeps(self, k):
        self._call(lib().mpr_set_fused_sweeps, int(k))

    def reset_chain(self, trial=0):
        self._call(lib().mpr_reset_chain, int(trial))

    # -- the path ------------------------------------------------------------------------
    def estimate_temperature(self):
        T, es, nt = C.c_double(), C.c_double(), C.c_int()
        self._call(lib().mpr_estimate_temperature, C.byref(T), C.byref(es), C.byref(nt))
        return T.value, es.value, nt.value

    def run(self, n_eq, n_meas, want_pred=True):
        """Returns (pred CUDA tensor [L, L] or None, e_mean, e_stderr)."""
        pred = self._torch.empty(self.shape, dtype=self._torch.float64, device=self.device) if want_pred else None
        m, s = C.c_double(), C.c_double()
        self._call(lib().mpr_run, int(n_eq), int(n_meas), pred.data_ptr() if want_pred else None,
                   C.byref(m), C.byref(s))
        return pred, m.value, s.value

    def sweep(self, n=1):
        self._call(lib().mpr_sweep, int(n))

    def pass_(self, kind, colour, sweep=0):
        self._call(lib().mpr_pass, PASS_KINDS[kind] if isinstance(kind, str) else int(kind), int(colour), int(sweep))

    # -- inspection ----------------------------------------------------------------------
    def get_state(self):
        phi = self._torch.empty(self.shape, dtype=self._torch.float64, device=self.device)
        self._call(lib().mpr_get_state, phi.data_ptr())
        return phi

    def set_state(self, phi):
        phi = self._torch.as_tensor(phi, dtype=self._torch.float64).to(self.device).contiguous()
        assert tuple(phi.shape) == self.shape
        self._call(lib().mpr_set_state, phi.data_ptr())
        self._torch.cuda.synchronize(self.device)

    def energy(self):
        H, e = C.c_double(), C.c_double()
        self._call(lib().mpr_energy, C.byref(H), C.byref(e))
        return H.value, e.value

    def sample_energy(self):
        es, n = C.c_double(), C.c_int64()
        self._call(lib().mpr_sample_energy, C.byref(es), C.byref(n))
        return es.value, n.value

    def counters(self):
        a, b, c = C.c_uint64(), C.c_uint64(), C.c_uint64()
        self._call(lib().mpr_get_counters, C.byref(a), C.byref(b), C.byref(c))
        return a.value, b.value, c.value

    def series(self):
        n = lib().mpr_get_energy_series(self.h, None, 0)
        out = np.empty(max(int(n), 0), dtype=np.float64)
        if n > 0:
            lib().mpr_get_energy_series(self.h, out.ctypes.data_as(C.POINTER(C.c_double)), n)
        return out

    def info(self):
        a, b, n, T = C.c_double(), C.c_double(), C.c_int64(), C.c_double()
        self._call(lib().mpr_get_info, C.byref(a), C.byref(b), C.byref(n), C.byref(T))
        return {"z_min": a.value, "z_max": b.value, "n_free": n.value, "T": T.value}

    def run_timing(self):
        """(device ms, launches, sweeps) of the equilibration phase of the last run() -- mpr_get_run_timing."""
        ms, nl, ns = C.c_double(), C.c_int64(), C.c_int64()
        self._call(lib().mpr_get_run_timing, C.byref(ms), C.byref(nl), C.byref(ns))
        return ms.value, nl.value, ns.value

    # -- slabs of a larger grid (include/mpr.h, "Slabs"; orchestrated by slabs.py) -------------
    def set_slab(self, global_row0, own_begin, own_end, z_min, z_max, global_bonds):
        self._call(lib().mpr_set_slab, int(global_row0), int(own_begin), int(own_end), float(z_min), float(z_max),
                   float(global_bonds))

    def set_peers(self, up, down):
        """Peer mode (mpr_set_peers): up / down = the Mpr objects of the slabs above / below, or None."""
        self._call(lib().mpr_set_peers, up.h if up is not None else None, down.h if down is not None else None)

    def sample_energy_parts(self):
        s, n = C.c_double(), C.c_int64()
        self._call(lib().mpr_sample_energy_parts, C.byref(s), C.byref(n))
        return s.value, n.value

    def rows_bytes(self, n_rows):
        n = C.c_size_t()
        self._call(lib().mpr_rows_bytes, int(n_rows), C.byref(n))
        return n.value

    def export_rows(self, row_begin, n_rows, out=None):
        """n_rows rows of the chain state from row_begin on -> uint8 CUDA tensor of rows_bytes(n_rows)."""
        if out is None:
            out = self._torch.empty(self.rows_bytes(n_rows), dtype=self._torch.uint8, device=self.device)
        self._call(lib().mpr_export_rows, int(row_begin), int(n_rows), out.data_ptr())
        return out

    def import_rows(self, row_begin, n_rows, buf):
        assert buf.is_cuda and buf.is_contiguous() and buf.numel() == self.rows_bytes(n_rows)
        self._call(lib().mpr_import_rows, int(row_begin), int(n_rows), buf.data_ptr())

    def advance(self, n_sweeps, measure=0, first_slot=0):
        self._call(lib().mpr_advance, int(n_sweeps), int(measure), int(first_slot))

    def quench(self, n_double_passes):
        self._call(lib().mpr_quench, int(n_double_passes))

    def fetch_series(self, n):
        out = np.empty(int(n), dtype=np.float64)
        self._call(lib().mpr_fetch_series, int(n), out.ctypes.data_as(C.POINTER(C.c_double)))
        return out

    def predict(self):
        pred = self._torch.empty(self.shape, dtype=self._torch.float64, device=self.device)
        self._call(lib().mpr_predict, pred.data_ptr())
        return pred

    def launches(self):
        n = C.c_uint64()
        self._call(lib().mpr_get_launch_stats, C.byref(n))
        return n.value


def predict_host(values, mask, mode="DP", seed=0, T=-1.0, n_eq=100, n_meas=100, workspace=None, pred_out=None,
                 device="cuda:0"):
    """End-to-end call on HOST arrays (mpr_predict_host): host->device copies, create, (estimate T,)
    run, device->host copy of the prediction.  Returns (pred numpy [L, L], e_mean, e_stderr, T, launches)."""
    torch = _torch()
    values = np.ascontiguousarray(values, dtype=np.float64)
    mask = np.ascontiguousarray(mask, dtype=np.uint8)
    Ly, Lx = int(mask.shape[0]), int(mask.shape[1])
    assert values.shape == mask.shape
    dev = torch.device(device)
    if workspace is None:
        workspace = torch.empty(workspace_bytes((Ly, Lx), host=True) + 256, dtype=torch.uint8, device=dev)
    off = (-workspace.data_ptr()) % 256
    if pred_out is None:
        pred_out = np.empty((Ly, Lx), dtype=np.float64)
    m, s, Tu, nl = C.c_double(), C.c_double(), C.c_double(), C.c_uint64()
    with torch.cuda.device(dev):
        tail = (values.ctypes.data, mask.ctypes.data, MODES[mode], int(seed), float(T), int(n_eq), int(n_meas),
                workspace.data_ptr() + off, workspace.numel() - off, torch.cuda.current_stream(dev).cuda_stream,
                pred_out.ctypes.data, C.byref(m), C.byref(s), C.byref(Tu), C.byref(nl))
        st = lib().mpr_predict_host(Lx, *tail) if Lx == Ly else lib().mpr_predict_host_rect(Lx, Ly, *tail)
    if st != MPR_OK:
        raise MprError(st)
    return pred_out, m.value, s.value, Tu.value, nl.value


def debug_trial_lengths():
    """(equilibration sweeps, measurement sweeps) of one temperature trial of R6, as the library runs it."""
    a, b = C.c_int(), C.c_int()
    lib().mpr_debug_trial_lengths(C.byref(a), C.byref(b))
    return a.value, b.value


def static_max_sites():
    return int(lib().mpr_static_max_sites())


def sample_energy_static(d_values, d_mask, out, q=0.5, stream=None, shape=None):
    """mpr_sample_energy_static: the sample energy and range of (d_values, d_mask) -- CUDA tensors f64 / u8 of shape
    (Ly, Lx) -- into `out` (CUDA f64[6]: e_s, pairs, z_min, z_max, measured sites, non-finite values), enqueued on
    `stream` (default: torch's current stream).  Argument marshalling only: no tensor is created here and the library
    allocates nothing.  `shape` overrides the tensors' shape (for the size checks)."""
    torch = _torch()
    Ly, Lx = shape if shape is not None else (int(d_mask.shape[0]), int(d_mask.shape[1]))
    dev = d_mask.device
    sptr = stream.cuda_stream if stream is not None else torch.cuda.current_stream(dev).cuda_stream
    with torch.cuda.device(dev):
        st = lib().mpr_sample_energy_static(int(Lx), int(Ly), d_values.data_ptr(), d_mask.data_ptr(), float(q), sptr,
                                            out.data_ptr())
    if st != MPR_OK:
        raise MprError(st, lib().mpr_static_last_error().decode())
    return out


def debug_proposal_width(T, q=None):
    return lib().mpr_debug_proposal_width(float(T)) if q is None else lib().mpr_debug_proposal_width_q(float(T), float(q))


def debug_series_stats(series):
    """(mean, binned standard error) of a host series by the library's own routine (R16).  No GPU needed."""
    v = np.ascontiguousarray(series, dtype=np.float64)
    m, s = C.c_double(), C.c_double()
    st = lib().mpr_debug_series_stats(v.ctypes.data_as(C.POINTER(C.c_double)), len(v), C.byref(m), C.byref(s))
    if st != MPR_OK:
        raise MprError(st)
    return m.value, s.value


def debug_match_temperature(e_sample, energy_of_T):
    """The library's R6 root search driven by a Python function T -> (e, se).  No GPU needed.
    Returns (T_hat, [trial temperatures in order])."""
    asked = []

    def cb(T, idx, e, se, _user):
        asked.append(T)
        e[0], se[0] = energy_of_T(T)
        return 0

    T, n = C.c_double(), C.c_int()
    st = lib().mpr_debug_match_temperature(float(e_sample), TRIAL_FN(cb), None, C.byref(T), C.byref(n))
    if st != MPR_OK:
        err = MprError(st)
        err.asked = asked
        raise err
    assert n.value == len(asked)
    return T.value, asked


def debug_accept(words, mdE, T, device="cuda:0"):
    """mpr_debug_accept: words uint32 [n, 2], mdE float64 [n] -> uint8 [n] (bit 0 filtered, bit 1 plain, bit 2 fast)."""
    torch = _torch()
    dev = torch.device(device)
    words = np.ascontiguousarray(words, dtype=np.uint32).reshape(-1, 2)
    mdE = np.ascontiguousarray(mdE, dtype=np.float64).reshape(-1)
    assert words.shape[0] == mdE.shape[0]
    d_w = torch.from_numpy(words.view(np.int32)).to(dev)
    d_e = torch.from_numpy(mdE).to(dev)
    out = torch.empty(mdE.shape[0], dtype=torch.uint8, device=dev)
    with torch.cuda.device(dev):
        st = lib().mpr_debug_accept(d_w.data_ptr(), d_e.data_ptr(), float(T), out.data_ptr(), mdE.shape[0],
                                    torch.cuda.current_stream(dev).cuda_stream)
    if st != MPR_OK:
        raise MprError(st)
    return out.cpu().numpy()


def debug_philox(ctr, key, device="cuda:0"):
    """Philox4x32-10 as the kernels evaluate it, for n counters: ctr uint32 [n, 4], key (k0, k1)."""
    torch = _torch()
    dev = torch.device(device)
    ctr = np.ascontiguousarray(ctr, dtype=np.uint32).reshape(-1, 4)
    d_ctr = torch.from_numpy(ctr.view(np.int32)).to(dev)
    d_out = torch.empty_like(d_ctr)
    k = (C.c_uint32 * 2)(int(key[0]) & 0xFFFFFFFF, int(key[1]) & 0xFFFFFFFF)
    with torch.cuda.device(dev):
        st = lib().mpr_debug_philox(d_ctr.data_ptr(), k, d_out.data_ptr(), ctr.shape[0],
                                    torch.cuda.current_stream(dev).cuda_stream)
    if st != MPR_OK:
        raise MprError(st)
    torch.cuda.synchronize(dev)
    return d_out.cpu().numpy().view(np.uint32)
