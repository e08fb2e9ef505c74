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


def test_rows_options_and_plan_argument_errors(L):
    """kbmod_search_rows / kbmod_plan_create / kbmod_search_planned / kbmod_search_host reject bad
    bands, options and shapes before any launch (no device here: a valid call would return -5)."""
    f = np.zeros(64, np.float32)
    buf = np.zeros(4096, np.uint8)
    fp = ctypes.c_void_p((f.ctypes.data + 15) // 16 * 16)
    ws = ctypes.c_void_p((buf.ctypes.data + 255) // 256 * 256)
    t = np.array([0.0, 1.0]).ctypes.data_as(ctypes.c_void_p)
    vel = np.ones(2, np.float32).ctypes.data_as(ctypes.c_void_p)

    class R(ctypes.Structure):
        _fields_ = [(n, ctypes.c_void_p) for n in ("a", "b", "c", "d", "e", "f")]

    class O(ctypes.Structure):
        _fields_ = [(n, ctypes.c_int32) for n in ("struct_size", "kernel", "tile_group_w", "staged_geom")]
    r = R(*[f.ctypes.data] * 6)
    big = ctypes.c_size_t(1 << 40)
    rows = lambda y0, y1, opt=None: L.kbmod_search_rows(fp, t, 2, 4, 4, vel, 1, 1, 1, y0, y1, ctypes.byref(r), ws, big,
                                                        ctypes.byref(opt) if opt else None, None)
    assert rows(-1, 2) == -3 and rows(3, 2) == -3 and rows(0, 5) == -3            # band outside [0, H]
    assert rows(0, 4, O(16, 9, 0, 0)) == -3 and rows(0, 4, O(16, -1, 0, 0)) == -3  # unknown kernel
    assert rows(0, 4, O(16, 0, 300, 0)) == -3 and rows(0, 4, O(16, 3, 0, 4)) == -3 # knobs out of range
    assert rows(0, 4, O(12, 0, 0, 0)) == -3                                         # wrong struct_size
    assert L.kbmod_search_rows(fp, t, 2, 4, 4, vel, 1, 1, 1, 0, 4, ctypes.byref(r), ws, ctypes.c_size_t(8), None, None) == -7
    # plans: host objects, no device needed
    h = ctypes.c_void_p()
    assert L.kbmod_plan_create(t, 2, 4, 4, vel, 1, 1, None, None) == -1
    assert L.kbmod_plan_create(t, 2, 4, 4, vel, 1, 33, None, ctypes.byref(h)) == -6 and not h
    assert L.kbmod_plan_create(t, 2, 0, 4, vel, 1, 1, None, ctypes.byref(h)) == -2
    bad_t = np.array([0.0, np.inf]).ctypes.data_as(ctypes.c_void_p)
    assert L.kbmod_plan_create(bad_t, 2, 4, 4, vel, 1, 1, None, ctypes.byref(h)) == -3
    assert L.kbmod_plan_create(t, 2, 4, 4, vel, 1, 1, None, ctypes.byref(h)) == 0 and h
    assert L.kbmod_plan_kernel(h) == 2                       # automatic resolves to the tiled kernel
    assert L.kbmod_search_planned(h, fp, 3, 0, 4, ctypes.byref(r), ws, big, None) == -3     # min_obs > N
    assert L.kbmod_search_planned(h, fp, 1, 2, 1, ctypes.byref(r), ws, big, None) == -3     # bad band
    assert L.kbmod_search_planned(h, None, 1, 0, 4, ctypes.byref(r), ws, big, None) == -1
    L.kbmod_plan_destroy(h)
    L.kbmod_plan_destroy(None)
    for k, want in ((1, 1), (3, 3), (4, 4)):
        h = ctypes.c_void_p()
        o = O(16, k, 0, 0)
        assert L.kbmod_plan_create(t, 2, 4, 4, vel, 1, 1, ctypes.byref(o), ctypes.byref(h)) == 0
        assert L.kbmod_plan_kernel(h) == want
        L.kbmod_plan_destroy(h)
    # a shape beyond the tiled kernel: automatic falls back to the direct kernel, explicit 2 is refused
    h = ctypes.c_void_p()
    assert L.kbmod_plan_create(t, 2, 40000, 4, vel, 1, 1, None, ctypes.byref(h)) == 0 and L.kbmod_plan_kernel(h) == 1
    L.kbmod_plan_destroy(h)
    o = O(16, 2, 0, 0)
    assert L.kbmod_plan_create(t, 2, 40000, 4, vel, 1, 1, ctypes.byref(o), ctypes.byref(h)) == -6
    # kbmod_search_host: the search-stage errors are reported before anything is enqueued
    psf = np.ones(1, np.float32).ctypes.data_as(ctypes.c_void_p)
    host = lambda K, mo, P: L.kbmod_search_host(fp, fp, None, psf, t, 2, 4, 4, P, vel, 1, K, mo, ctypes.byref(r), ws,
                                                big, None, None)
    assert host(40, 1, 1) == -6 and host(1, 3, 1) == -3 and host(1, 1, 2) == -3 and host(1, 1, 33) == -6


def test_no_cpu_fallback_without_device(L):
    import torch
    if torch.cuda.is_available():
        pytest.skip("device present")
    buf = np.zeros(4096, np.float32)
    p = ctypes.c_void_p((buf.ctypes.data + 255) // 256 * 256)
    one = np.ones(1, np.float32).ctypes.data_as(ctypes.c_void_p)
    assert L.kbmod_make_psi_phi(p, p, None, one, 1, 2, 2, 1, p, None) == -5


def test_next_row_calls_reject_bad_arguments_before_any_launch(L):
    """kbmod_search_threshold / kbmod_filter_candidates / kbmod_coadd_stamps / kbmod_build_mask /
    kbmod_cluster_candidates: every argument error has its code and is found before a device is
    needed (no GPU here: a call that passes all checks returns KBMOD_ERR_CUDA = -5)."""
    import torch
    f = np.zeros(256, np.float32)
    buf = np.zeros(8192, np.uint8)
    fp = ctypes.c_void_p((f.ctypes.data + 15) // 16 * 16)
    ws = ctypes.c_void_p((buf.ctypes.data + 255) // 256 * 256)
    t = np.array([0.0, 1.0]).ctypes.data_as(ctypes.c_void_p)
    bad_t = np.array([0.0, np.nan]).ctypes.data_as(ctypes.c_void_p)
    vel = np.ones(2, np.float32).ctypes.data_as(ctypes.c_void_p)
    big = ctypes.c_size_t(1 << 40)
    cf = ctypes.c_float
    no_gpu = -5 if not torch.cuda.is_available() else 0

    class C(ctypes.Structure):
        _fields_ = [(n, ctypes.c_void_p) for n in ("x", "y", "v", "n", "psi", "phi", "nu", "alpha")]
    c = C(*[f.ctypes.data] * 8)
    thr = lambda mo=1, nu=cf(5.0), y0=0, y1=4, cap=4, cnt=fp, opt=None, wsb=big: L.kbmod_search_threshold(
        fp, t, 2, 4, 4, vel, 1, mo, nu, y0, y1, ctypes.byref(c), ctypes.c_longlong(cap), cnt, ws, wsb, opt, None)
    assert thr(mo=3) == -3 and thr(nu=cf(float("nan"))) == -3 and thr(y0=3, y1=2) == -3 and thr(cap=-1) == -3
    assert thr(cnt=None) == -1 and thr(wsb=ctypes.c_size_t(16)) == -7

    class O(ctypes.Structure):
        _fields_ = [(n, ctypes.c_int32) for n in ("struct_size", "kernel", "tile_group_w", "staged_geom")]
    assert thr(opt=ctypes.byref(O(16, 2, 0, 0))) == -6 and thr(opt=ctypes.byref(O(16, 3, 0, 0))) == -6   # top-K only kernels
    if no_gpu:
        assert thr() == no_gpu and thr(opt=ctypes.byref(O(16, 4, 0, 0))) == no_gpu

    filt = lambda N=2, M=1, s=cf(5.0), q=cf(0.0), tt=t, xy=fp: L.kbmod_filter_candidates(
        fp, tt, N, 4, 4, xy, fp, M, s, q, fp, fp, fp, fp, fp, fp, None, None)
    assert filt(N=65) == -6 and filt(N=0) == -2 and filt(M=-1) == -2 and filt(s=cf(0.0)) == -3
    assert filt(q=cf(-1.0)) == -3 and filt(tt=bad_t) == -3 and filt(xy=None) == -1
    if no_gpu:
        assert filt() == no_gpu

    stamps = lambda R=3, M=1, N=2: L.kbmod_coadd_stamps(fp, None, t, N, 4, 4, fp, fp, None, M, R, fp, None, None)
    assert stamps(R=-1) == -3 and stamps(R=16) == -6 and stamps(N=65) == -6 and stamps(M=-2) == -2
    if no_gpu:
        assert stamps() == no_gpu

    mask = lambda grow=2, mi=2, out=fp: L.kbmod_build_mask(fp, fp, None, 2, 4, 4, cf(5.0), grow, mi, cf(120.0), out, None)
    assert mask(grow=-1) == -3 and mask(grow=9) == -6 and mask(mi=0) == -3 and mask(out=None) == -1
    if no_gpu:
        assert mask() == no_gpu

    L.kbmod_cluster_workspace.restype = ctypes.c_size_t
    assert L.kbmod_cluster_workspace(1000) >= 1000 * 9 and L.kbmod_cluster_workspace(-1) == 0
    clus = lambda M=4, exy=cf(2.0), ev=cf(4.0), ms=1, wsb=big: L.kbmod_cluster_candidates(
        fp, fp, fp, M, exy, ev, ms, fp, fp, ws, wsb, None)
    assert clus(M=-1) == -2 and clus(exy=cf(0.0)) == -3 and clus(ev=cf(float("inf"))) == -3 and clus(ms=0) == -3
    assert clus(wsb=ctypes.c_size_t(8)) == -7
    if no_gpu:
        assert clus() == no_gpu and clus(M=0) == no_gpu
