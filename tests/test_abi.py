"""CPU-side checks of the boundary: libmpr.so builds, loads and exports every symbol that
include/mpr.h declares; argument validation that needs no GPU."""
import ctypes as C
import os
import re

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def mpr_mod():
    from paper_1910_08448_b200 import build, mpr
    build.build()
    mpr.lib()
    return mpr


def declared_symbols():
    with open(os.path.join(ROOT, "include", "mpr.h")) as fh:
        text = fh.read()
    text = re.sub(r"/\*.*?\*/", "", text, flags=re.S)
    return sorted(set(re.findall(r"\b(mpr_[a-z_0-9]+)\s*\(", text)))


def test_header_symbols_are_exported(mpr_mod):
    syms = declared_symbols()
    assert len(syms) >= 25
    lib = C.CDLL(mpr_mod.LIB_PATH)
    for s in syms:
        assert hasattr(lib, s), s
    assert sorted(mpr_mod.SYMBOLS) == syms


def test_workspace_bytes_and_status_strings(mpr_mod):
    assert mpr_mod.workspace_bytes(64) > 2 * 2 * 64 * 32 * 16
    assert mpr_mod.workspace_bytes(16384) < 16 * 2 ** 30
    assert mpr_mod.workspace_bytes(64, host=True) >= mpr_mod.workspace_bytes(64) + 17 * 64 * 64
    with pytest.raises(mpr_mod.MprError) as ei:
        mpr_mod.workspace_bytes(1)
    assert ei.value.code == mpr_mod.ERR_INVALID_ARG
    lib = mpr_mod.lib()
    assert lib.mpr_status_string(0) == b"ok"
    assert b"CUDA" in lib.mpr_status_string(mpr_mod.ERR_CUDA)


def test_create_rejects_bad_arguments_without_gpu(mpr_mod):
    lib = mpr_mod.lib()
    h = C.c_void_p()
    assert lib.mpr_create(C.byref(h), 1, None, None, None, 0, None) == mpr_mod.ERR_INVALID_ARG
    assert lib.mpr_create(C.byref(h), 8, 256, 256, None, 1 << 30, None) == mpr_mod.ERR_WORKSPACE
    assert lib.mpr_create(C.byref(h), 8, 256, 256, 256, 1024, None) == mpr_mod.ERR_WORKSPACE     # too small
    assert lib.mpr_create(C.byref(h), 8, 256, 256, 257, 1 << 30, None) == mpr_mod.ERR_WORKSPACE
    assert not h.value


def test_no_cpu_fallback(mpr_mod):
    """Without a CUDA device the product path must fail loudly, not compute on the CPU."""
    import torch
    if torch.cuda.is_available():
        pytest.skip("GPU present")
    import numpy as np
    with pytest.raises(RuntimeError):
        mpr_mod.Mpr(np.zeros((8, 8)), np.zeros((8, 8), dtype=np.uint8))


def test_product_does_not_import_oracle():
    """The CUDA package neither imports, links nor loads anything under oracle/."""
    pkg = os.path.join(ROOT, "paper_1910_08448_b200")
    for dirpath, _, files in os.walk(pkg):
        for f in files:
            if f.endswith((".py", ".cu", ".cuh", ".h")):
                with open(os.path.join(dirpath, f)) as fh:
                    text = fh.read()
                for needle in ("import oracle", "from oracle", "mpr_oracle", "oracle/", "oracle."):
                    assert needle not in text, (f, needle)
