"""CPU oracle of the KBMOD shift-and-stack hot path (TEST INFRASTRUCTURE ONLY).

Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs
may import this package.  It shares nothing with paper_1901_02492_b200/ (the CUDA path).
The arithmetic lives in oracle.c (plain C, written from PAPER.md); this file only builds
the shared object with gcc and marshals numpy arrays into it.
"""
from __future__ import annotations

import ctypes
import os
import subprocess
from typing import Optional

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "oracle.c")
# KBMOD_ORACLE_SANITIZE=1 (tests/test_simt_sanitized.py, in a child interpreter that preloads the ASan
# runtime): the same source built with -fsanitize=address,undefined into its own shared object
_SANITIZE = os.environ.get("KBMOD_ORACLE_SANITIZE") == "1"
_LIB = os.path.join(_HERE, "liboracle_asan.so" if _SANITIZE else "liboracle.so")
_lib: Optional[ctypes.CDLL] = None

MODE_F64 = 0
MODE_F32SEQ = 1


def build(force: bool = False) -> str:
    """gcc -O2 -ffp-contract=off -fopenmp; rebuilt when oracle.c is newer than the .so."""
    if (not force and os.path.exists(_LIB)
            and os.path.getmtime(_LIB) >= os.path.getmtime(_SRC)):
        return _LIB
    san = ["-g", "-fno-omit-frame-pointer", "-fsanitize=address,undefined",
           "-fno-sanitize-recover=all"] if _SANITIZE else []
    cmd = ["gcc", "-O2", "-std=c99", "-ffp-contract=off", "-fno-fast-math", "-fopenmp", *san,
           "-shared", "-fPIC", "-o", _LIB, _SRC, "-lm"]
    subprocess.run(cmd, check=True)
    return _LIB


def lib() -> ctypes.CDLL:
    global _lib
    if _lib is None:
        _lib = ctypes.CDLL(build())
        _lib.oracle_num_threads.restype = ctypes.c_int
        for name in ("oracle_make_psi_phi", "oracle_search", "oracle_eval_all",
                     "oracle_eval_trajectories", "oracle_score"):
            getattr(_lib, name).restype = ctypes.c_int
    return _lib


def num_threads() -> int:
    return int(lib().oracle_num_threads())


def set_threads(n: int) -> None:
    lib().oracle_set_threads(ctypes.c_int(int(n)))


def _p(a: Optional[np.ndarray]):
    return None if a is None else a.ctypes.data_as(ctypes.c_void_p)


def _c(a, dtype):
    return np.ascontiguousarray(a, dtype=dtype)


def make_psi_phi(sci, var, mask, psf, want_abs: bool = False):
    """-> psiphi [N,H,W,2] f32 (and psi_abs [N,H,W] f32 if want_abs)."""
    sci = _c(sci, np.float32)
    var = _c(var, np.float32)
    psf = _c(psf, np.float32)
    N, H, W = sci.shape
    P = psf.shape[-1]
    assert var.shape == sci.shape and psf.shape == (N, P, P)
    if mask is not None:
        mask = _c(mask, np.uint8)
        assert mask.shape == sci.shape
    out = np.empty((N, H, W, 2), dtype=np.float32)
    pabs = np.empty((N, H, W), dtype=np.float32) if want_abs else None
    rc = lib().oracle_make_psi_phi(_p(sci), _p(var), _p(mask), _p(psf), N, H, W, P,
                                   _p(out), _p(pabs))
    if rc != 0:
        raise ValueError(f"oracle_make_psi_phi failed: {rc}")
    return (out, pabs) if want_abs else out


def search(psiphi, times, vel_grid, K, min_obs, mode=MODE_F32SEQ, y_begin=0, y_end=None):
    """-> dict of planes [(y_end-y_begin), W, K]: vel_idx,n_obs (i32), psi,phi,nu,alpha (f32)."""
    psiphi = _c(psiphi, np.float32)
    times = _c(times, np.float64)
    vel = _c(vel_grid, np.float32)
    N, H, W, _ = psiphi.shape
    V = vel.shape[0]
    y_end = H if y_end is None else y_end
    rows = y_end - y_begin
    res = {
        "vel_idx": np.empty((rows, W, K), np.int32), "n_obs": np.empty((rows, W, K), np.int32),
        "psi": np.empty((rows, W, K), np.float32), "phi": np.empty((rows, W, K), np.float32),
        "nu": np.empty((rows, W, K), np.float32), "alpha": np.empty((rows, W, K), np.float32),
    }
    rc = lib().oracle_search(_p(psiphi), _p(times), N, H, W, _p(vel), V, int(K), int(min_obs),
                             int(mode), int(y_begin), int(y_end),
                             _p(res["vel_idx"]), _p(res["n_obs"]), _p(res["psi"]),
                             _p(res["phi"]), _p(res["nu"]), _p(res["alpha"]))
    if rc != 0:
        raise ValueError(f"oracle_search failed: {rc}")
    return res


def eval_all(psiphi, times, vel_grid, mode=MODE_F32SEQ, y_begin=0, y_end=None):
    """-> Psi, Phi [rows,W,V] f32, n_obs [rows,W,V] i32."""
    psiphi = _c(psiphi, np.float32)
    times = _c(times, np.float64)
    vel = _c(vel_grid, np.float32)
    N, H, W, _ = psiphi.shape
    V = vel.shape[0]
    y_end = H if y_end is None else y_end
    rows = y_end - y_begin
    Psi = np.empty((rows, W, V), np.float32)
    Phi = np.empty((rows, W, V), np.float32)
    nobs = np.empty((rows, W, V), np.int32)
    rc = lib().oracle_eval_all(_p(psiphi), _p(times), N, H, W, _p(vel), V, int(mode),
                               int(y_begin), int(y_end), _p(Psi), _p(Phi), _p(nobs))
    if rc != 0:
        raise ValueError(f"oracle_eval_all failed: {rc}")
    return Psi, Phi, nobs


def eval_trajectories(psiphi, times, x0y0, vxvy, mode=MODE_F32SEQ):
    """-> Psi, Phi [M] f32, n_obs [M] i32, ixiy [M,N,2] i32."""
    psiphi = _c(psiphi, np.float32)
    times = _c(times, np.float64)
    x0y0 = _c(x0y0, np.int32).reshape(-1, 2)
    vxvy = _c(vxvy, np.float32).reshape(-1, 2)
    N, H, W, _ = psiphi.shape
    M = x0y0.shape[0]
    assert vxvy.shape[0] == M
    Psi = np.empty(M, np.float32)
    Phi = np.empty(M, np.float32)
    nobs = np.empty(M, np.int32)
    ixiy = np.empty((M, N, 2), np.int32)
    rc = lib().oracle_eval_trajectories(_p(psiphi), _p(times), N, H, W, _p(x0y0), _p(vxvy), M,
                                        int(mode), _p(Psi), _p(Phi), _p(nobs), _p(ixiy))
    if rc != 0:
        raise ValueError(f"oracle_eval_trajectories failed: {rc}")
    return Psi, Phi, nobs, ixiy


def score(Psi, Phi):
    """S5 on arrays -> nu, alpha (f32, correctly rounded)."""
    Psi = _c(Psi, np.float32)
    Phi = _c(Phi, np.float32)
    nu = np.empty_like(Psi)
    alpha = np.empty_like(Psi)
    rc = lib().oracle_score(_p(Psi), _p(Phi), ctypes.c_size_t(Psi.size), _p(nu), _p(alpha))
    if rc != 0:
        raise ValueError(f"oracle_score failed: {rc}")
    return nu, alpha


# ----------------------------------------------------------------------------- next rows (N1..N4)
def search_threshold(psiphi, times, vel_grid, min_obs, nu_min, y_begin=0, y_end=None, capacity=1 << 22):
    """N4 -> (count, dict of arrays [min(count, capacity)]: x, y, vel_idx, n_obs, psi, phi, nu, alpha),
    in (y0, x0, j) order."""
    psiphi = _c(psiphi, np.float32)
    times = _c(times, np.float64)
    vel = _c(vel_grid, np.float32)
    N, H, W, _ = psiphi.shape
    y_end = H if y_end is None else y_end
    ints = {k: np.zeros(capacity, np.int32) for k in ("x", "y", "vel_idx", "n_obs")}
    flts = {k: np.zeros(capacity, np.float32) for k in ("psi", "phi", "nu", "alpha")}
    fn = lib().oracle_search_threshold
    fn.restype = ctypes.c_longlong
    n = fn(_p(psiphi), _p(times), N, H, W, _p(vel), int(vel.shape[0]), int(min_obs), ctypes.c_float(nu_min),
           int(y_begin), int(y_end), ctypes.c_longlong(capacity), _p(ints["x"]), _p(ints["y"]),
           _p(ints["vel_idx"]), _p(ints["n_obs"]), _p(flts["psi"]), _p(flts["phi"]), _p(flts["nu"]),
           _p(flts["alpha"]))
    if n < 0:
        raise ValueError(f"oracle_search_threshold failed: {n}")
    k = min(int(n), capacity)
    return int(n), {**{a: v[:k] for a, v in ints.items()}, **{a: v[:k] for a, v in flts.items()}}


def filter_candidates(psiphi, times, x0y0, vxvy, sigma_reject=5.0, q=0.0):
    """N1 -> dict: psi, phi, nu, alpha [M] f32, n_obs [M] i32, keep [M] u64, kalman [M,2] f32."""
    psiphi = _c(psiphi, np.float32)
    times = _c(times, np.float64)
    x0y0 = _c(x0y0, np.int32).reshape(-1, 2)
    vxvy = _c(vxvy, np.float32).reshape(-1, 2)
    N, H, W, _ = psiphi.shape
    M = x0y0.shape[0]
    out = {k: np.zeros(M, np.float32) for k in ("psi", "phi", "nu", "alpha")}
    out["n_obs"] = np.zeros(M, np.int32)
    out["keep"] = np.zeros(M, np.uint64)
    out["kalman"] = np.zeros((M, 2), np.float32)
    lib().oracle_filter_candidates.restype = ctypes.c_int
    rc = lib().oracle_filter_candidates(_p(psiphi), _p(times), N, H, W, _p(x0y0), _p(vxvy), M,
                                        ctypes.c_float(sigma_reject), ctypes.c_float(q), _p(out["psi"]),
                                        _p(out["phi"]), _p(out["n_obs"]), _p(out["nu"]), _p(out["alpha"]),
                                        _p(out["keep"]), _p(out["kalman"]))
    if rc != 0:
        raise ValueError(f"oracle_filter_candidates failed: {rc}")
    return out


def build_mask(sci, var, mask_in=None, sigma_thr=5.0, grow=2, min_images=2, bright_counts=120.0):
    """N3 -> mask [N,H,W] u8."""
    sci = _c(sci, np.float32)
    var = _c(var, np.float32)
    N, H, W = sci.shape
    if mask_in is not None:
        mask_in = _c(mask_in, np.uint8)
    out = np.zeros((N, H, W), np.uint8)
    lib().oracle_build_mask.restype = ctypes.c_int
    rc = lib().oracle_build_mask(_p(sci), _p(var), _p(mask_in), N, H, W, ctypes.c_float(sigma_thr), int(grow),
                                 int(min_images), ctypes.c_float(bright_counts), _p(out))
    if rc != 0:
        raise ValueError(f"oracle_build_mask failed: {rc}")
    return out


def coadd_stamps(sci, mask, times, x0y0, vxvy, keep=None, R=10):
    """N2 -> stamps [M,2R+1,2R+1] f32, moments [M,6] f32 (m00, cx, cy, mu20, mu02, mu11)."""
    sci = _c(sci, np.float32)
    times = _c(times, np.float64)
    x0y0 = _c(x0y0, np.int32).reshape(-1, 2)
    vxvy = _c(vxvy, np.float32).reshape(-1, 2)
    N, H, W = sci.shape
    M = x0y0.shape[0]
    if mask is not None:
        mask = _c(mask, np.uint8)
    if keep is not None:
        keep = _c(keep, np.uint64)
    S = 2 * R + 1
    stamps = np.zeros((M, S, S), np.float32)
    moments = np.zeros((M, 6), np.float32)
    lib().oracle_coadd_stamps.restype = ctypes.c_int
    rc = lib().oracle_coadd_stamps(_p(sci), _p(mask), _p(times), N, H, W, _p(x0y0), _p(vxvy), _p(keep), M, int(R),
                                   _p(stamps), _p(moments))
    if rc != 0:
        raise ValueError(f"oracle_coadd_stamps failed: {rc}")
    return stamps, moments


def cluster_candidates(x0y0, vxvy, nu, eps_xy=2.0, eps_v=4.0, min_samples=1):
    """N5 -> label [M] i32 (smallest core index of the cluster, -1 = noise), rep [M] u8."""
    x0y0 = _c(x0y0, np.int32).reshape(-1, 2)
    vxvy = _c(vxvy, np.float32).reshape(-1, 2)
    nu = _c(nu, np.float32)
    M = x0y0.shape[0]
    label = np.zeros(M, np.int32)
    rep = np.zeros(M, np.uint8)
    lib().oracle_cluster_candidates.restype = ctypes.c_int
    rc = lib().oracle_cluster_candidates(_p(x0y0), _p(vxvy), _p(nu), M, ctypes.c_float(eps_xy), ctypes.c_float(eps_v),
                                         int(min_samples), _p(label), _p(rep))
    if rc != 0:
        raise ValueError(f"oracle_cluster_candidates failed: {rc}")
    return label, rep
