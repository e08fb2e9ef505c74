"""CPU-only checks of the C-ABI library: it loads, exports every symbol the header declares,
and rejects bad arguments before touching a device (no compute calls here)."""
import ctypes
import os
import re

import numpy as np
import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def L():
    from paper_1901_02492_b200 import build, binding
    build.build()
    return binding.lib()


def _header_symbols():
    src = open(os.path.join(ROOT, "include", "kbmod_b200.h")).read()
    src = re.sub(r"/\*.*?\*/", "", src, flags=re.S)
    return sorted(set(re.findall(r"\b(kbmod_[a-z_]+)\s*\(", src)))


def test_exports_every_declared_symbol(L):
    from paper_1901_02492_b200 import binding
    syms = _header_symbols()
    assert len(syms) >= 9
    for s in syms:
        assert hasattr(L, s), s
    assert sorted(binding.EXPORTS) == syms


def test_pure_functions(L):
    assert L.kbmod_version().decode() .count(".") == 1
    assert L.kbmod_status_string(0) == b"ok"
    assert L.kbmod_status_string(-6) != L.kbmod_status_string(-5)
    n = L.kbmod_search_workspace(15, 4096, 4096, 640, 8)
    assert n >= 15 * 4096 * 4096 * 8
    assert L.kbmod_search_workspace(0, 1, 1, 1, 1) == 0


def test_argument_errors_before_any_launch(L):
    f = np.zeros(16, np.float32)
    fp = f.ctypes.data_as(ctypes.c_void_p)
    t = np.zeros(2, np.float64).ctypes.data_as(ctypes.c_void_p)
    assert L.kbmod_make_psi_phi(None, fp, None, fp, 1, 2, 2, 1, fp, None) == -1
    assert L.kbmod_make_psi_phi(fp, fp, None, fp, 1, 0, 2, 1, fp, None) == -2
    assert L.kbmod_make_psi_phi(fp, fp, None, fp, 1, 2, 2, 2, fp, None) == -3
    assert L.kbmod_make_psi_phi(fp, fp, None, fp, 1, 2, 2, 33, fp, None) == -6

    class R(ctypes.Structure):
        _fields_ = [(n, ctypes.c_void_p) for n in ("a", "b", "c", "d", "e", "f")]
    r = R(*[f.ctypes.data] * 6)
    assert L.kbmod_search(None, t, 2, 2, 2, fp, 1, 1, 1, ctypes.byref(r), fp, 0, None) == -1
    assert L.kbmod_search(fp, t, 2, 2, 2, fp, 1, 33, 1, ctypes.byref(r), fp, 0, None) == -6
    assert L.kbmod_search(fp, t, 2, 2, 2, fp, 1, 1, 3, ctypes.byref(r), fp, 0, None) == -3
    assert L.kbmod_search(fp, t, 65, 2, 2, fp, 1, 1, 1, ctypes.byref(r), fp, 0, None) == -6
    assert L.kbmod_set_search_kernel(7) == -3
    assert L.kbmod_set_search_kernel(0) == 0


def test_no_cpu_fallback_without_device(L):
    import torch
    if torch.cuda.is_available():
        pytest.skip("device present")
    buf = np.zeros(4096, np.float32)
    p = ctypes.c_void_p((buf.ctypes.data + 255) // 256 * 256)
    one = np.ones(1, np.float32).ctypes.data_as(ctypes.c_void_p)
    assert L.kbmod_make_psi_phi(p, p, None, one, 1, 2, 2, 1, p, None) == -5
