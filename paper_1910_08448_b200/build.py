"""Builds libmpr.so (the C-ABI CUDA library) in-tree with nvcc for sm_100a.

    python -m paper_1910_08448_b200.build [--force]

Eight translation units compiled in parallel: mpr.cu (C ABI, host logic, PLAIN and TILED kernels), mpr_static.cu (the
entry point that needs no workspace) and
mpr_strip_mode.cu once per precision mode (the STRIP kernels), then one device link into the shared library.
"""
from __future__ import annotations

import os
import subprocess
import sys
from concurrent.futures import ThreadPoolExecutor

_HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(_HERE, "csrc")
OBJ = os.path.join(_HERE, "build")
LIB = os.path.join(_HERE, "libmpr.so")
HEADERS = ["mpr_device.cuh", "mpr_host_math.hpp", "mpr_plain.cuh", "mpr_tiled.cuh", "mpr_strip.cuh",
           os.path.join("..", "..", "include", "mpr.h")]
# (source, object name, extra flags)
UNITS = [("mpr.cu", "mpr.o", []), ("mpr_static.cu", "mpr_static.o", [])] + \
        [("mpr_strip_mode.cu", "mpr_strip_mode%d.o" % m, ["-DMPR_STRIP_MODE=%d" % m]) for m in range(6)]

NVCC_FLAGS = [
    "-gencode", "arch=compute_100a,code=sm_100a",
    "-O3", "-std=c++17", "-lineinfo",
    "--fmad=false",            # every fused multiply-add is written out in the sources (bit-identical paths)
    "-Xcompiler", "-fPIC",
    "-Xptxas", "-v",
]


def _stale() -> bool:
    if not os.path.exists(LIB):
        return True
    t = os.path.getmtime(LIB)
    deps = [os.path.join(CSRC, f) for f in [u[0] for u in UNITS] + HEADERS] + [os.path.abspath(__file__)]
    return any(os.path.getmtime(d) > t for d in deps)


def build(force: bool = False, verbose: bool = False) -> str:
    if not (force or _stale()):
        return LIB
    nvcc = os.environ.get("NVCC", "nvcc")
    os.makedirs(OBJ, exist_ok=True)

    def compile_unit(u):
        src, obj, extra = u
        cmd = [nvcc] + NVCC_FLAGS + extra + ["-c", "-o", os.path.join(OBJ, obj), os.path.join(CSRC, src)]
        res = subprocess.run(cmd, capture_output=True, text=True)
        return cmd, res

    with ThreadPoolExecutor(max_workers=len(UNITS)) as ex:
        results = list(ex.map(compile_unit, UNITS))
    link = [nvcc, "-gencode", "arch=compute_100a,code=sm_100a", "-shared", "-Xcompiler", "-fPIC", "-o", LIB] + \
           [os.path.join(OBJ, u[1]) for u in UNITS]
    log = os.path.join(_HERE, "build.log")
    ok = all(r.returncode == 0 for _, r in results)
    lres = subprocess.run(link, capture_output=True, text=True) if ok else None
    with open(log, "w") as fh:
        for cmd, r in results:
            fh.write(" ".join(cmd) + "\n" + r.stdout + r.stderr)
        if lres is not None:
            fh.write(" ".join(link) + "\n" + lres.stdout + lres.stderr)
    if verbose or not ok or (lres is not None and lres.returncode != 0):
        for _, r in results:
            sys.stderr.write(r.stdout + r.stderr)
        if lres is not None:
            sys.stderr.write(lres.stdout + lres.stderr)
    if not ok or lres.returncode != 0:
        raise RuntimeError("nvcc failed building libmpr.so (see %s)" % log)
    return LIB


if __name__ == "__main__":
    print(build(force="--force" in sys.argv, verbose=True))
