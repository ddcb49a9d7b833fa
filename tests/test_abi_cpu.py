"""CPU-only checks of the boundary: the C-ABI library loads, exports every symbol the header declares,
validates arguments before touching CUDA, and fails loudly (no fallback) without a device."""
import ctypes
import os
import re

import numpy as np
import pytest

from paper_2205_00856_b200 import binding as B
from paper_2205_00856_b200 import build as build_mod

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def lib():
    build_mod.build_library()
    return B.lib()


def header_symbols():
    src = open(os.path.join(ROOT, "include", "cn_nshape.h")).read()
    src = re.sub(r"/\*.*?\*/", "", src, flags=re.S)
    return sorted(set(re.findall(r"\b(cn_[a-z_]+)\s*\((?!\*)", src)))  # (not the function-pointer typedef)


def test_exports_every_declared_symbol(lib):
    syms = header_symbols()
    assert set(syms) == set(B.EXPORTS), (syms, B.EXPORTS)
    for s in syms:
        assert hasattr(lib, s), s


def test_status_strings(lib):
    for code in range(6):
        assert lib.cn_status_string(code).decode().startswith("CN_")
    assert B.cn_version().startswith("cn_nshape")


@pytest.mark.parametrize("N,P,dx,dt", [(1, 1, 0.1, 0.1), (8, 0, 0.1, 0.1), (8, 9, 0.1, 0.1), (8, 2, 0.0, 0.1),
                                       (8, 2, -1.0, 0.1), (8, 2, 0.1, 0.0), (8, 2, float("nan"), 0.1),
                                       (8, 2, 0.1, float("inf"))])
def test_invalid_arguments_rejected_before_cuda(lib, N, P, dx, dt):
    V = np.zeros(max(N, 1))
    h = ctypes.c_void_p()
    st = lib.cn_plan_create(ctypes.byref(h), N, P, dx, dt, V.ctypes.data)
    assert st == B.CN_EINVAL and not h.value


def test_null_pointers(lib):
    assert lib.cn_plan_create(None, 8, 2, 0.1, 0.1, None) == B.CN_EINVAL
    h = ctypes.c_void_p()
    assert lib.cn_plan_create(ctypes.byref(h), 8, 2, 0.1, 0.1, None) == B.CN_EINVAL
    assert lib.cn_factorize(None, None) == B.CN_EINVAL
    assert lib.cn_step(None, None, 1, None) == B.CN_EINVAL
    assert lib.cn_destroy(None) == B.CN_EINVAL
    assert lib.cn_batched_sweep(None, None, 1, 1, 1, 1, None) == B.CN_EINVAL


def test_no_cpu_fallback(lib):
    import torch
    if torch.cuda.is_available():
        pytest.skip("CUDA device present")
    V = np.zeros(64)
    with pytest.raises(B.CnError) as ei:
        B.cn_plan_create(64, 8, 0.1, 0.01, V)
    assert ei.value.status in (B.CN_ECUDA, B.CN_ENOMEM)


def test_product_does_not_import_oracle():
    pkg = os.path.join(ROOT, "paper_2205_00856_b200")
    for dirpath, _, files in os.walk(pkg):
        for f in files:
            if f.endswith((".py", ".cu", ".cuh", ".h")):
                txt = open(os.path.join(dirpath, f)).read()
                assert not re.search(r"^\s*(from|import)\s+oracle", txt, flags=re.M), f
                assert "cn_oracle" not in txt and "cn_thomas" not in txt, f
    for f in os.listdir(os.path.join(ROOT, "oracle")):
        if f.endswith((".py", ".c")):
            txt = open(os.path.join(ROOT, "oracle", f)).read()
            assert not re.search(r"^\s*(from|import)\s+paper_2205_00856_b200", txt, flags=re.M), f
