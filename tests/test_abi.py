"""C-ABI boundary checks that need no GPU: the library loads, exports every symbol include/ts_b200.h declares, the
binding lists the same symbols, and argument errors are reported as statuses (no compute call is made here)."""
import ctypes
import os
import re

import numpy as np
import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
HEADER = os.path.join(ROOT, "include", "ts_b200.h")


def declared_symbols():
    src = open(HEADER).read()
    src = re.sub(r"/\*.*?\*/", "", src, flags=re.S)
    return sorted(set(re.findall(r"\b(ts_[a-z0-9_]+)\s*\(", src)))


@pytest.fixture(scope="module")
def lib():
    from paper_1305_0036_b200 import build, binding
    build.build()
    return binding.load()


def test_header_declares_the_four_north_star_calls():
    syms = declared_symbols()
    for name in ("ts_create", "ts_set_state", "ts_evolve", "ts_expect"):
        assert name in syms


def test_library_exports_every_declared_symbol(lib):
    from paper_1305_0036_b200 import binding
    syms = declared_symbols()
    assert sorted(binding.SYMBOLS) == syms, "binding.SYMBOLS and include/ts_b200.h disagree"
    for name in syms:
        assert hasattr(lib, name), name


def test_signatures_hold_no_torch_types():
    src = open(HEADER).read()
    assert "torch" not in src.lower().replace("pytorch", "") and "at::" not in src and "Tensor" not in src


def test_status_strings(lib):
    from paper_1305_0036_b200 import binding as B
    assert B.strerror(B.TS_OK) == "ok"
    for st in (B.TS_ERR_ARG, B.TS_ERR_NOMEM, B.TS_ERR_CUDA, B.TS_ERR_NOSTATE):
        assert B.strerror(st) not in ("ok", "unknown status")
    assert B.strerror(-99) == "unknown status"
    assert "sm_100a" in B.version()


def test_argument_errors_are_statuses_not_crashes(lib):
    from paper_1305_0036_b200 import binding as B
    ctx = ctypes.c_void_p()
    dp = ctypes.POINTER(ctypes.c_double)
    h = np.zeros((3, 4)); J = np.zeros((3, 4, 4))
    hp, Jp = h.ctypes.data_as(dp), J.ctypes.data_as(dp)
    assert lib.ts_create(None, 4, hp, Jp) == B.TS_ERR_ARG
    assert lib.ts_create(ctypes.byref(ctx), 0, hp, Jp) == B.TS_ERR_ARG
    assert lib.ts_create(ctypes.byref(ctx), 34, hp, Jp) == B.TS_ERR_ARG
    assert lib.ts_create(ctypes.byref(ctx), 4, None, Jp) == B.TS_ERR_ARG
    hbad = h.copy(); hbad[1, 2] = np.nan
    assert lib.ts_create(ctypes.byref(ctx), 4, hbad.ctypes.data_as(dp), Jp) == B.TS_ERR_ARG
    assert not ctx.value
    # NULL contexts
    assert lib.ts_destroy(None) == B.TS_OK
    assert lib.ts_evolve(None, 0.01, 1, 4) == B.TS_ERR_ARG
    out = ctypes.c_double()
    assert lib.ts_expect(None, 2, 0, ctypes.byref(out)) == B.TS_ERR_ARG
    assert lib.ts_norm2(None, ctypes.byref(out)) == B.TS_ERR_ARG


def test_no_cpu_fallback_without_a_device(lib):
    """On a box without a GPU, ts_create reports TS_ERR_CUDA and the Python class raises: the product path never
    computes on the CPU."""
    import torch
    if torch.cuda.is_available():
        pytest.skip("a CUDA device is present")
    from paper_1305_0036_b200 import binding as B
    ctx = ctypes.c_void_p()
    dp = ctypes.POINTER(ctypes.c_double)
    h = np.zeros((3, 4)); J = np.zeros((3, 4, 4))
    assert lib.ts_create(ctypes.byref(ctx), 4, h.ctypes.data_as(dp), J.ctypes.data_as(dp)) == B.TS_ERR_CUDA
    with pytest.raises(RuntimeError):
        B.TrotterSuzuki(4, h, J)


def test_product_path_does_not_import_the_oracle():
    pkg = os.path.join(ROOT, "paper_1305_0036_b200")
    for dirpath, _, files in os.walk(pkg):
        for f in files:
            if f.endswith((".py", ".cu", ".cuh", ".h")):
                txt = open(os.path.join(dirpath, f)).read()
                assert "ts_oracle" not in txt, f
                assert not re.search(r"^\s*(from|import)\s+oracle\b", txt, flags=re.M), f
    ora = os.path.join(ROOT, "oracle")
    for f in os.listdir(ora):
        if f.endswith((".py", ".c", ".h")):
            txt = open(os.path.join(ora, f)).read()
            assert not re.search(r"^\s*(from|import)\s+paper_1305_0036_b200\b", txt, flags=re.M), f
            assert "#include \"../paper" not in txt and "libts_b200" not in txt, f
