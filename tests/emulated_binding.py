"""TEST INFRASTRUCTURE: the interface of paper_1901_02492_b200.binding served by the SIMT-emulated
library (tests/hostlogic/*_simt.cpp: the product's own launch code and kernels compiled with g++)
on CPU tensors.  It exists so that the LOGIC of the `-m gpu` test files -- their cases, their
expectations, their use of the API -- can be exercised on a machine without a GPU
(`KBMOD_GPU_TESTS_EMULATED=1 pytest -m gpu ...`, and tests/test_gpu_tests_emulated.py in the CPU
suite): a GPU test that is wrong fails here, not on the first B200 that runs it.  It proves nothing
about hardware.  Not part of the product; the product has no CPU path.
"""
import ctypes

import numpy as np
import torch

from tests import simt_build

PLANES = ("vel_idx", "n_obs", "psi", "phi", "nu", "alpha")
_CAND_I, _CAND_F = ("x", "y", "vel_idx", "n_obs"), ("psi", "phi", "nu", "alpha")
KERNEL_AUTO, KERNEL_DIRECT, KERNEL_TILED, KERNEL_STAGED, KERNEL_TILED_QUEUED = range(5)
_default_kernel = 0
_launches = 0
_libs = {}


class KbmodError(RuntimeError):
    pass


def _lib(name):
    if name not in _libs:
        _libs[name] = simt_build.load(name)
    return _libs[name]


def lib():
    return _lib("tiled_simt")


def launch_count():
    return _launches


def set_search_kernel(which):
    global _default_kernel
    if not 0 <= int(which) <= 4:
        raise KbmodError(f"unknown search kernel {which}")
    _default_kernel = int(which)


def _np(t, dtype):
    a = t.detach().numpy() if isinstance(t, torch.Tensor) else np.asarray(t)
    return np.ascontiguousarray(a, dtype=dtype)


def _p(a):
    return None if a is None else a.ctypes.data_as(ctypes.c_void_p)


class Plan:
    def __init__(self, times, N, H, W, vel_grid, K, kernel=None, tile_group_w=0, staged_geom=0):
        self.times, self.vel = _np(times, np.float64), _np(vel_grid, np.float32)
        self.N, self.H, self.W, self.V, self.K = N, H, W, self.vel.shape[0], K
        self.kernel = _default_kernel if kernel is None else kernel
        self.kernel = 2 if self.kernel == 0 else self.kernel
        self.tile_group_w, self.staged_geom = tile_group_w, staged_geom

    def close(self):
        pass


def alloc_result(H, W, K, device=None):
    r = {k: torch.empty((H, W, K), dtype=torch.int32) for k in PLANES[:2]}
    r.update({k: torch.empty((H, W, K), dtype=torch.float32) for k in PLANES[2:]})
    return r


def search_workspace(N, H, W, V, K):
    return 256


def search_status(workspace):
    return None


def make_psi_phi(sci, var, mask, psf, out=None):
    global _launches
    s, v = _np(sci, np.float32), _np(var, np.float32)
    m = None if mask is None else _np(mask, np.uint8)
    psf = _np(psf, np.float32)
    N, H, W = s.shape
    if psf.ndim != 3 or psf.shape[0] != N or psf.shape[1] != psf.shape[2]:
        raise KbmodError("psf must be [N,P,P]")
    res = np.zeros((N, H, W, 2), np.float32)
    n = ctypes.c_int(0)
    rc = _lib("post_simt").simt_make_psi_phi(_p(s), _p(v), _p(m), _p(psf), N, H, W, psf.shape[-1], _p(res), 0,
                                             ctypes.byref(n), 2, ctypes.c_uint(3))
    if rc:
        raise KbmodError(f"kbmod_make_psi_phi failed: {rc}")
    _launches += n.value
    t = torch.from_numpy(res)
    if out is not None:
        out.copy_(t)
        return out
    return t


def search(psiphi, times, vel_grid, K, min_obs, out=None, workspace=None, y_begin=0, y_end=None, kernel=None,
           tile_group_w=0, staged_geom=0, plan=None):
    global _launches
    if not isinstance(psiphi, torch.Tensor):
        raise KbmodError("psiphi: expected a tensor")
    pp = _np(psiphi, np.float32)
    N, H, W, _ = pp.shape
    if plan is not None:
        times, vel_grid, kernel, tile_group_w, staged_geom = plan.times, plan.vel, plan.kernel, plan.tile_group_w, plan.staged_geom
    t, vel = _np(times, np.float64), _np(vel_grid, np.float32)
    y_end = H if y_end is None else int(y_end)
    k = _default_kernel if kernel is None else int(kernel)
    if K > 32 or N > 64:
        raise KbmodError("kbmod_search_rows failed: -6 (beyond the supported limits)")
    if K < 1 or min_obs < 1 or min_obs > N or not np.isfinite(t).all() or not (0 <= y_begin <= y_end <= H):
        raise KbmodError("kbmod_search_rows failed: -3 (argument out of range)")
    res = {p: np.zeros((y_end - y_begin, W, K), np.int32 if p in PLANES[:2] else np.float32) for p in PLANES}
    args = (_p(pp), _p(t), N, H, W, _p(vel), int(vel.shape[0]), int(K), int(min_obs), int(y_begin), y_end,
            *[_p(res[p]) for p in PLANES])
    stats = (ctypes.c_longlong * 8)()
    if k == KERNEL_DIRECT:
        rc = _lib("post_simt").simt_search_direct(*args, 2, ctypes.c_uint(5))
    elif k == KERNEL_STAGED:
        rc = _lib("staged_simt").simt_search_staged(*args, int(staged_geom), 2, ctypes.c_uint(5), 3, 7, stats)
        if stats[0] or stats[2] or stats[4]:
            raise KbmodError("emulated staged kernel reported a fault")
    else:
        rc = _lib("tiled_simt").simt_search_tiled(*args, int(k == KERNEL_TILED_QUEUED), int(tile_group_w), 2,
                                                  ctypes.c_uint(5), stats)
    if rc:
        raise KbmodError(f"kbmod_search_rows failed: {rc}")
    _launches += 2
    got = {p: torch.from_numpy(a) for p, a in res.items()}
    if out is not None:
        for p in PLANES:
            out[p].copy_(got[p])
        return out
    return got


def eval_trajectories(psiphi, times, x0y0, vxvy, want_pixels=True):
    pp = _np(psiphi, np.float32)
    N, H, W, _ = pp.shape
    xy, v = _np(x0y0, np.int32), _np(vxvy, np.float32)
    M = xy.shape[0]
    Psi, Phi, n = np.zeros(M, np.float32), np.zeros(M, np.float32), np.zeros(M, np.int32)
    ix = np.zeros((M, N, 2), np.int32)
    rc = _lib("post_simt").simt_eval_trajectories(_p(pp), _p(_np(times, np.float64)), N, H, W, _p(xy), _p(v), M,
                                                  _p(Psi), _p(Phi), _p(n), _p(ix) if want_pixels else None)
    if rc:
        raise KbmodError(f"kbmod_eval_trajectories failed: {rc}")
    return tuple(torch.from_numpy(a) for a in (Psi, Phi, n)) + ((torch.from_numpy(ix),) if want_pixels else (None,))


def search_threshold(psiphi, times, vel_grid, min_obs, nu_min, capacity, y_begin=0, y_end=None, kernel=None,
                     tile_group_w=0, workspace=None):
    pp = _np(psiphi, np.float32)
    N, H, W, _ = pp.shape
    t, vel = _np(times, np.float64), _np(vel_grid, np.float32)
    y_end = H if y_end is None else int(y_end)
    cap = max(1, int(capacity))
    out = {k: np.zeros(cap, np.int32) for k in _CAND_I}
    out.update({k: np.zeros(cap, np.float32) for k in _CAND_F})
    k = _default_kernel if kernel is None else int(kernel)
    libn, fn = ("tiled_simt", "simt_search_tiled_threshold") if k == KERNEL_TILED_QUEUED else ("post_simt", "simt_search_direct_threshold")
    f = getattr(_lib(libn), fn)
    f.restype = ctypes.c_longlong
    n = f(_p(pp), _p(t), N, H, W, _p(vel), int(vel.shape[0]), int(min_obs), ctypes.c_float(nu_min), int(y_begin), y_end,
          ctypes.c_longlong(int(capacity)), *[_p(out[c]) for c in _CAND_I + _CAND_F], 2, ctypes.c_uint(5))
    if n < 0:
        raise KbmodError(f"kbmod_search_threshold failed: {n}")
    return torch.tensor([n], dtype=torch.int64), {c: torch.from_numpy(a) for c, a in out.items()}


def filter_candidates(psiphi, times, x0y0, vxvy, sigma_reject=5.0, process_var=0.0):
    pp = _np(psiphi, np.float32)
    N, H, W, _ = pp.shape
    xy, v = _np(x0y0, np.int32), _np(vxvy, np.float32)
    M = xy.shape[0]
    out = {k: np.zeros(M, np.float32) for k in ("psi", "phi", "nu", "alpha")}
    out["n_obs"], out["keep"], out["kalman"] = np.zeros(M, np.int32), np.zeros(M, np.int64), np.zeros((M, 2), np.float32)
    rc = _lib("post_simt").simt_filter_candidates(_p(pp), _p(_np(times, np.float64)), N, H, W, _p(xy), _p(v), M,
                                                  ctypes.c_float(sigma_reject), ctypes.c_float(process_var),
                                                  *[_p(out[k]) for k in ("psi", "phi", "n_obs", "nu", "alpha", "keep", "kalman")],
                                                  2, ctypes.c_uint(1))
    if rc:
        raise KbmodError(f"kbmod_filter_candidates failed: {rc}")
    return {k: torch.from_numpy(a) for k, a in out.items()}


def coadd_stamps(sci, mask, times, x0y0, vxvy, keep=None, R=10):
    s = _np(sci, np.float32)
    N, H, W = s.shape
    m = None if mask is None else _np(mask, np.uint8)
    xy, v = _np(x0y0, np.int32), _np(vxvy, np.float32)
    kp = None if keep is None else _np(keep, np.int64)
    M, S = xy.shape[0], 2 * int(R) + 1
    st, mo = np.zeros((M, S, S), np.float32), np.zeros((M, 6), np.float32)
    rc = _lib("post_simt").simt_coadd_stamps(_p(s), _p(m), _p(_np(times, np.float64)), N, H, W, _p(xy), _p(v), _p(kp), M,
                                             int(R), _p(st), _p(mo), 2, ctypes.c_uint(1))
    if rc:
        raise KbmodError(f"kbmod_coadd_stamps failed: {rc}")
    return torch.from_numpy(st), torch.from_numpy(mo)


def build_mask(sci, var, mask_in=None, sigma_thr=5.0, grow=2, min_images=2, bright_counts=120.0):
    s, v = _np(sci, np.float32), _np(var, np.float32)
    N, H, W = s.shape
    m = None if mask_in is None else _np(mask_in, np.uint8)
    out = np.zeros((N, H, W), np.uint8)
    rc = _lib("post_simt").simt_build_mask(_p(s), _p(v), _p(m), N, H, W, ctypes.c_float(sigma_thr), int(grow),
                                           int(min_images), ctypes.c_float(bright_counts), _p(out), 1, ctypes.c_uint(1))
    if rc:
        raise KbmodError(f"kbmod_build_mask failed: {rc}")
    return torch.from_numpy(out)


def cluster_candidates(x0y0, vxvy, nu, eps_xy=2.0, eps_v=4.0, min_samples=1):
    xy, v, n_ = _np(x0y0, np.int32), _np(vxvy, np.float32), _np(nu, np.float32)
    M = xy.shape[0]
    label, rep, n = np.zeros(M, np.int32), np.zeros(M, np.uint8), ctypes.c_int(0)
    rc = _lib("post_simt").simt_cluster_candidates(_p(xy), _p(v), _p(n_), M, ctypes.c_float(eps_xy), ctypes.c_float(eps_v),
                                                   int(min_samples), _p(label), _p(rep), ctypes.byref(n), 2, ctypes.c_uint(1))
    if rc:
        raise KbmodError(f"kbmod_cluster_candidates failed: {rc}")
    return torch.from_numpy(label), torch.from_numpy(rep)
