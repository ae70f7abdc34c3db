"""CPU-side checks of the boundary: the C-ABI library builds, loads and exports every symbol that
include/muser.h declares, the Python binding mirrors it, and the library's own host-side table generators
(A0) agree with the oracle's (DESIGN.md pin P5: library-vs-oracle tables).  No compute call needs a GPU here."""
import ctypes
import os
import re

import numpy as np
import pytest

from oracle import muser_oracle as mo
from paper_1712_06913_b200 import binding, build

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def lib():
    build.build()
    return binding.lib()


def _declared_symbols():
    text = open(os.path.join(ROOT, "include", "muser.h")).read()
    text = re.sub(r"/\*.*?\*/", "", text, flags=re.S)
    return sorted(set(re.findall(r"\b(muser_[a-z_0-9]+)\s*\(", text)))


def test_library_exports_every_declared_symbol(lib):
    names = _declared_symbols()
    assert len(names) >= 20
    raw = ctypes.CDLL(binding.LIB_PATH)
    for n in names:
        assert hasattr(raw, n), f"{n} declared in muser.h but not exported"
    assert sorted(binding.SIGNATURES) == names, "binding.SIGNATURES must mirror muser.h exactly"


def test_binding_has_no_oracle_or_cpu_fallback():
    pkg = os.path.join(ROOT, "paper_1712_06913_b200")
    for dirpath, _, files in os.walk(pkg):
        for fn in files:
            if fn.endswith((".py", ".cu", ".cpp", ".h")):
                src = open(os.path.join(dirpath, fn)).read()
                assert "import oracle" not in src and "from oracle" not in src, fn
                assert "oracle_c" not in src and "muser_oracle" not in src, fn


def test_create_without_gpu_fails_loudly(lib):
    import torch
    if torch.cuda.is_available():
        pytest.skip("GPU present")
    h = lib.muser_imager_create(256, 256, 10.0, 7, 8)
    assert not h
    assert b"no CPU fallback" in lib.muser_last_error(None)


@pytest.mark.parametrize("args", [(255, 256, 10.0, 7, 8), (256, 256, 10.0, 6, 8), (256, 256, 10.0, 7, 7),
                                  (256, 256, -1.0, 7, 8), (12, 256, 10.0, 7, 8), (256, 256, 10.0, 65, 8)])
def test_create_rejects_bad_arguments(lib, args):
    assert not lib.muser_imager_create(*args)
    assert len(lib.muser_last_error(None)) > 0


@pytest.mark.parametrize("S,Q", [(7, 128), (7, 8), (5, 64), (9, 32)])
def test_host_pswf_table_matches_oracle(lib, S, Q):
    T = binding.host_table(binding.MUSER_KERNEL_PSWF, S, Q)
    assert np.abs(T - mo.table_pswf(S, Q)).max() < 1e-12
    assert np.array_equal(T, T[::-1])            # exactly symmetric by construction
    assert T[S * Q // 2] == 1.0


def test_host_gauss_table_and_corrector_match_oracle(lib):
    T = binding.host_table(binding.MUSER_KERNEL_GAUSS, 7, 8, 0.0)
    assert np.abs(T - mo.table_gauss(7, 8, 1.55)).max() < 1e-15
    Tp = binding.host_table(binding.MUSER_KERNEL_PSWF, 7, 128)
    for n in (256, 1024):
        c = binding.host_corrector(Tp, 7, 128, n)
        assert np.abs(c / mo.corrector(mo.table_pswf(7, 128), 7, 128, n) - 1).max() < 1e-10


def test_host_wkernel_matches_oracle(lib):
    fov = 4096 * 2.5 * mo.ARCSEC
    for S, w in ((7, 0.0), (15, 6000.0), (31, 19900.0)):
        a = binding.host_wtable(S, 64, w, fov)
        b = mo.table_wkernel(S, 64, w, fov)
        assert np.abs(a - b).max() < 1e-12


def test_host_helpers_reject_bad_arguments(lib):
    out = np.zeros(100)
    assert lib.muser_host_table(0, 6, 8, 0.0, out.ctypes.data) == binding.MUSER_EINVAL
    assert lib.muser_host_table(7, 7, 8, 0.0, out.ctypes.data) == binding.MUSER_EINVAL
    assert lib.muser_host_table(0, 7, 8, 0.0, None) == binding.MUSER_EINVAL
    assert lib.muser_imager_destroy(None) == binding.MUSER_OK
    assert lib.muser_grid(None, None, None, None, None, 0, None) == binding.MUSER_EINVAL
