"""Thin Python binding of libkbmod_b200.so (include/kbmod_b200.h).

Argument marshalling only: every step of the path runs in the library's CUDA kernels.  PyTorch
supplies device memory and the stream.  There is no CPU fallback: if the library cannot be
loaded, or a compute call is made without a CUDA device, an exception is raised.
"""
from __future__ import annotations

import ctypes
import os
from typing import Dict, Optional

import numpy as np
import torch

_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(_HERE, "libkbmod_b200.so")
_lib: Optional[ctypes.CDLL] = None

EXPORTS = ("kbmod_make_psi_phi", "kbmod_search", "kbmod_search_rows", "kbmod_search_workspace",
           "kbmod_search_split", "kbmod_plan_create", "kbmod_plan_kernel", "kbmod_search_planned",
           "kbmod_plan_destroy", "kbmod_eval_trajectories", "kbmod_launch_count", "kbmod_status_string",
           "kbmod_version", "kbmod_debug_staged_plan", "kbmod_search_status", "kbmod_search_host",
           "kbmod_search_host_workspace", "kbmod_search_threshold", "kbmod_filter_candidates",
           "kbmod_coadd_stamps", "kbmod_build_mask", "kbmod_cluster_candidates", "kbmod_cluster_workspace")
_INT_CALLS = ("kbmod_cluster_candidates", "kbmod_search_threshold", "kbmod_filter_candidates", "kbmod_coadd_stamps", "kbmod_build_mask",
              "kbmod_make_psi_phi", "kbmod_search", "kbmod_search_rows", "kbmod_search_split",
              "kbmod_plan_create", "kbmod_plan_kernel", "kbmod_search_planned", "kbmod_eval_trajectories",
              "kbmod_debug_staged_plan", "kbmod_search_status", "kbmod_search_host")
KERNEL_AUTO, KERNEL_DIRECT, KERNEL_TILED, KERNEL_STAGED, KERNEL_TILED_QUEUED = range(5)


class KbmodError(RuntimeError):
    pass


class _Result(ctypes.Structure):
    _fields_ = [(n, ctypes.c_void_p) for n in ("vel_idx", "n_obs", "psi", "phi", "nu", "alpha")]


class _Candidates(ctypes.Structure):       # kbmod_candidates
    _fields_ = [(n, ctypes.c_void_p) for n in ("x", "y", "vel_idx", "n_obs", "psi", "phi", "nu", "alpha")]


class _Options(ctypes.Structure):          # kbmod_search_options
    _fields_ = [(n, ctypes.c_int32) for n in ("struct_size", "kernel", "tile_group_w", "staged_geom")]


# Default kernel of THIS MODULE's calls (a Python-side convenience for tests and benchmarks; the
# library itself has no process-wide setting: the choice travels in kbmod_search_options).
_default_kernel = KERNEL_AUTO


def _options(kernel=None, tile_group_w=0, staged_geom=0) -> _Options:
    k = _default_kernel if kernel is None else int(kernel)
    return _Options(ctypes.sizeof(_Options), k, int(tile_group_w), int(staged_geom))


def lib() -> ctypes.CDLL:
    """Loads the in-tree C-ABI library; raises if it has not been built (no fallback)."""
    global _lib
    if _lib is None:
        if not os.path.exists(LIB_PATH):
            raise KbmodError(f"{LIB_PATH} is missing: run paper_1901_02492_b200/build.py "
                             "(or __graft_entry__.build()); there is no CPU fallback")
        L = ctypes.CDLL(LIB_PATH)
        L.kbmod_search_workspace.restype = ctypes.c_size_t
        L.kbmod_search_host_workspace.restype = ctypes.c_size_t
        L.kbmod_cluster_workspace.restype = ctypes.c_size_t
        L.kbmod_launch_count.restype = ctypes.c_ulonglong
        L.kbmod_status_string.restype = ctypes.c_char_p
        L.kbmod_version.restype = ctypes.c_char_p
        for n in _INT_CALLS:
            getattr(L, n).restype = ctypes.c_int
        L.kbmod_plan_destroy.restype = None
        _lib = L
    return _lib


def _check(rc: int, what: str) -> None:
    if rc != 0:
        raise KbmodError(f"{what} failed: {rc} ({lib().kbmod_status_string(rc).decode()})")


def _dev(t: Optional[torch.Tensor], dtype, what: str):
    if t is None:
        return None
    if not (isinstance(t, torch.Tensor) and t.is_cuda and t.dtype == dtype and t.is_contiguous()):
        raise KbmodError(f"{what}: expected a contiguous CUDA tensor of {dtype}")
    return ctypes.c_void_p(t.data_ptr())


def _host(a, dtype) -> np.ndarray:
    if isinstance(a, torch.Tensor):
        a = a.detach().cpu().numpy()
    return np.ascontiguousarray(a, dtype=dtype)


def _stream() -> ctypes.c_void_p:
    return ctypes.c_void_p(torch.cuda.current_stream().cuda_stream)


def version() -> str:
    return lib().kbmod_version().decode()


def launch_count() -> int:
    return int(lib().kbmod_launch_count())


def set_search_kernel(which: int) -> None:
    """Sets the kernel this module passes in kbmod_search_options when a call names none."""
    global _default_kernel
    if not 0 <= int(which) <= 4:
        raise KbmodError(f"unknown search kernel {which}")
    _default_kernel = int(which)


class Plan:
    """kbmod_plan: the host plan of a search (times, velocity grid, shape, K, options), built once."""

    def __init__(self, times, N: int, H: int, W: int, vel_grid, K: int, kernel=None, tile_group_w=0,
                 staged_geom=0):
        t = _host(times, np.float64)
        v = _host(vel_grid, np.float32)
        if t.shape != (N,) or v.ndim != 2 or v.shape[1] != 2:
            raise KbmodError("times must be [N], vel_grid [V,2]")
        self.N, self.H, self.W, self.V, self.K = int(N), int(H), int(W), int(v.shape[0]), int(K)
        self._h = ctypes.c_void_p()
        opt = _options(kernel, tile_group_w, staged_geom)
        _check(lib().kbmod_plan_create(t.ctypes.data_as(ctypes.c_void_p), self.N, self.H, self.W,
                                       v.ctypes.data_as(ctypes.c_void_p), self.V, self.K, ctypes.byref(opt),
                                       ctypes.byref(self._h)), "kbmod_plan_create")

    @property
    def kernel(self) -> int:
        return int(lib().kbmod_plan_kernel(self._h))

    def close(self) -> None:
        if self._h:
            lib().kbmod_plan_destroy(self._h)
            self._h = ctypes.c_void_p()

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass


def search_status(workspace: torch.Tensor) -> None:
    """kbmod_search_status: synchronises the current stream and raises if the last search that
    used this workspace did not complete (KBMOD_ERR_TIMEOUT / CUDA fault)."""
    _check(lib().kbmod_search_status(_dev(workspace, torch.uint8, "workspace"), _stream()),
           "kbmod_search_status")


def debug_staged_plan(times, N: int, H: int, W: int, vel_grid, staged_geom: int = 0):
    """kbmod_debug_staged_plan (host only): returns (stream [nent, ints_per_entry] int32,
    shapes [nshapes, 2] int32, info dict)."""
    t = _host(times, np.float64)
    v = _host(vel_grid, np.float32).reshape(-1, 2)
    V = v.shape[0]
    B_guess = 8
    cap = (V // B_guess + 2) * (max(N - 1, 0) * B_guess + 1) * 128
    stream = np.zeros(cap, np.int32)
    shapes = np.zeros((4096, 2), np.int32)
    info = np.zeros(8, np.int32)
    rc = lib().kbmod_debug_staged_plan(t.ctypes.data_as(ctypes.c_void_p), N, H, W,
                                       v.ctypes.data_as(ctypes.c_void_p), V, int(staged_geom),
                                       stream.ctypes.data_as(ctypes.c_void_p), ctypes.c_size_t(cap),
                                       shapes.ctypes.data_as(ctypes.c_void_p), 4096,
                                       info.ctypes.data_as(ctypes.c_void_p))
    _check(rc, "kbmod_debug_staged_plan")
    keys = ("nent", "hdr_ints", "nshapes", "TW", "TH", "B", "CAP", "HDR_BYTES")
    d = {k: int(x) for k, x in zip(keys, info)}
    return stream[:d["nent"] * d["hdr_ints"]].reshape(d["nent"], d["hdr_ints"]).copy(), \
        shapes[:d["nshapes"]].copy(), d


def search_workspace(N: int, H: int, W: int, V: int, K: int) -> int:
    return int(lib().kbmod_search_workspace(N, H, W, V, K))


def alloc_workspace(nbytes: int, device) -> torch.Tensor:
    """Device scratch for the calls that take a workspace (256-byte alignment is required; the CUDA
    caching allocator aligns every block to 512 bytes)."""
    return torch.empty(int(nbytes), dtype=torch.uint8, device=device)


def make_psi_phi(sci: torch.Tensor, var: torch.Tensor, mask: Optional[torch.Tensor], psf,
                 out: Optional[torch.Tensor] = None) -> torch.Tensor:
    """kbmod_make_psi_phi: sci/var [N,H,W] f32 cuda, mask [N,H,W] u8 cuda or None, psf host
    [N,P,P] -> psiphi [N,H,W,2] f32 cuda."""
    N, H, W = sci.shape
    psf = _host(psf, np.float32)
    if psf.ndim != 3 or psf.shape[0] != N or psf.shape[1] != psf.shape[2]:
        raise KbmodError("psf must be [N,P,P]")
    if var.shape != sci.shape or (mask is not None and mask.shape != sci.shape):
        raise KbmodError("sci, var, mask shapes differ")
    if out is None:
        out = torch.empty((N, H, W, 2), dtype=torch.float32, device=sci.device)
    rc = lib().kbmod_make_psi_phi(_dev(sci, torch.float32, "sci"), _dev(var, torch.float32, "var"),
                                  _dev(mask, torch.uint8, "mask"),
                                  psf.ctypes.data_as(ctypes.c_void_p), N, H, W, psf.shape[1],
                                  _dev(out, torch.float32, "psiphi"), _stream())
    _check(rc, "kbmod_make_psi_phi")
    return out


def alloc_result(H: int, W: int, K: int, device) -> Dict[str, torch.Tensor]:
    r = {k: torch.empty((H, W, K), dtype=torch.int32, device=device) for k in ("vel_idx", "n_obs")}
    r.update({k: torch.empty((H, W, K), dtype=torch.float32, device=device)
              for k in ("psi", "phi", "nu", "alpha")})
    return r


def _result_struct(out: Dict[str, torch.Tensor], rows: int, W: int, K: int) -> _Result:
    for k in ("vel_idx", "n_obs", "psi", "phi", "nu", "alpha"):
        _dev(out[k], torch.int32 if k in ("vel_idx", "n_obs") else torch.float32, k)
        if tuple(out[k].shape) != (rows, W, K):
            raise KbmodError(f"result plane {k}: expected shape {(rows, W, K)}, got {tuple(out[k].shape)}")
    return _Result(*[ctypes.c_void_p(out[k].data_ptr()) for k in ("vel_idx", "n_obs", "psi", "phi", "nu", "alpha")])


def search(psiphi: torch.Tensor, times, vel_grid, K: int, min_obs: int,
           out: Optional[Dict[str, torch.Tensor]] = None,
           workspace: Optional[torch.Tensor] = None, y_begin: int = 0, y_end: Optional[int] = None,
           kernel: Optional[int] = None, tile_group_w: int = 0, staged_geom: int = 0,
           plan: Optional[Plan] = None) -> Dict[str, torch.Tensor]:
    """kbmod_search_rows (kbmod_search_planned when `plan` is given): psiphi [N,H,W,2] f32 cuda, times
    host [N] f64, vel_grid host [V,2] f32.  Searches the start rows [y_begin, y_end) (default: all);
    the result planes hold that band only, [(y_end - y_begin), W, K]."""
    N, H, W, two = psiphi.shape
    if two != 2:
        raise KbmodError("psiphi must be [N,H,W,2]")
    y_end = H if y_end is None else int(y_end)
    y_begin = int(y_begin)
    if plan is not None:
        if (plan.N, plan.H, plan.W, plan.K) != (N, H, W, int(K)):
            raise KbmodError("plan was built for another shape or K")
        V = plan.V
    else:
        times = _host(times, np.float64)
        vel = _host(vel_grid, np.float32)
        if times.shape != (N,) or vel.ndim != 2 or vel.shape[1] != 2:
            raise KbmodError("times must be [N], vel_grid [V,2]")
        V = vel.shape[0]
    rows = max(0, y_end - y_begin)
    if out is None:
        out = alloc_result(rows, W, K, psiphi.device)
    need = search_workspace(N, H, W, V, K)
    own_workspace = workspace is None
    if own_workspace:
        workspace = alloc_workspace(need, psiphi.device)
    res = _result_struct(out, rows, W, int(K))
    if plan is not None:
        rc = lib().kbmod_search_planned(plan._h, _dev(psiphi, torch.float32, "psiphi"), int(min_obs), y_begin,
                                        y_end, ctypes.byref(res), _dev(workspace, torch.uint8, "workspace"),
                                        ctypes.c_size_t(workspace.numel()), _stream())
        _check(rc, "kbmod_search_planned")
    else:
        opt = _options(kernel, tile_group_w, staged_geom)
        rc = lib().kbmod_search_rows(_dev(psiphi, torch.float32, "psiphi"),
                                     times.ctypes.data_as(ctypes.c_void_p), N, H, W,
                                     vel.ctypes.data_as(ctypes.c_void_p), V, int(K), int(min_obs), y_begin, y_end,
                                     ctypes.byref(res), _dev(workspace, torch.uint8, "workspace"),
                                     ctypes.c_size_t(workspace.numel()), ctypes.byref(opt), _stream())
        _check(rc, "kbmod_search_rows")
    if own_workspace:
        # convenience path (no caller workspace to query later): wait and report a kernel that
        # gave up; callers that pass a workspace stay asynchronous and call search_status()
        search_status(workspace)
    return out


def search_host_workspace(N: int, H: int, W: int, V: int, K: int) -> int:
    return int(lib().kbmod_search_host_workspace(N, H, W, V, K))


def _hostbuf(t, dtype, what: str):
    if t is None:
        return None
    if not (isinstance(t, torch.Tensor) and not t.is_cuda and t.dtype == dtype and t.is_contiguous()):
        raise KbmodError(f"{what}: expected a contiguous host tensor of {dtype} (pinned for async copies)")
    return ctypes.c_void_p(t.data_ptr())


def search_host(sci: torch.Tensor, var: torch.Tensor, mask: Optional[torch.Tensor], psf, times,
                vel_grid, K: int, min_obs: int, out: Dict[str, torch.Tensor],
                workspace: torch.Tensor, kernel: Optional[int] = None) -> Dict[str, torch.Tensor]:
    """kbmod_search_host: the whole hot path from HOST tensors (pinned for asynchronous copies) to
    HOST result planes `out`; `workspace` is a CUDA uint8 tensor of search_host_workspace() bytes.
    Enqueued on the current stream; synchronise it (or call search_status) before reading `out`."""
    N, H, W = sci.shape
    psf = _host(psf, np.float32)
    times = _host(times, np.float64)
    vel = _host(vel_grid, np.float32)
    if psf.ndim != 3 or psf.shape[0] != N or psf.shape[1] != psf.shape[2]:
        raise KbmodError("psf must be [N,P,P]")
    if tuple(var.shape) != (N, H, W) or (mask is not None and tuple(mask.shape) != (N, H, W)):
        raise KbmodError("sci, var, mask shapes differ")
    if times.shape != (N,) or vel.ndim != 2 or vel.shape[1] != 2:
        raise KbmodError("times must be [N], vel_grid [V,2]")
    for k in ("vel_idx", "n_obs", "psi", "phi", "nu", "alpha"):
        if tuple(out[k].shape) != (H, W, int(K)):
            raise KbmodError(f"result plane {k}: expected shape {(H, W, int(K))}, got {tuple(out[k].shape)}")
    if workspace.numel() < search_host_workspace(N, H, W, int(vel.shape[0]), int(K)):
        raise KbmodError("workspace smaller than search_host_workspace()")
    res = _Result(*[_hostbuf(out[k], torch.int32 if k in ("vel_idx", "n_obs") else torch.float32, k)
                    for k in ("vel_idx", "n_obs", "psi", "phi", "nu", "alpha")])
    opt = _options(kernel)
    rc = lib().kbmod_search_host(_hostbuf(sci, torch.float32, "sci"), _hostbuf(var, torch.float32, "var"),
                                 _hostbuf(mask, torch.uint8, "mask"), psf.ctypes.data_as(ctypes.c_void_p),
                                 times.ctypes.data_as(ctypes.c_void_p), N, H, W, int(psf.shape[1]),
                                 vel.ctypes.data_as(ctypes.c_void_p), int(vel.shape[0]), int(K), int(min_obs),
                                 ctypes.byref(res), _dev(workspace, torch.uint8, "workspace"),
                                 ctypes.c_size_t(workspace.numel()), ctypes.byref(opt), _stream())
    _check(rc, "kbmod_search_host")
    return out


def search_split(psi: torch.Tensor, phi: torch.Tensor, times, vel_grid, K: int, min_obs: int):
    """kbmod_search_split: psi, phi as separate [N,H,W] f32 cuda planes."""
    N, H, W = psi.shape
    times = _host(times, np.float64)
    vel = _host(vel_grid, np.float32)
    V = vel.shape[0]
    out = alloc_result(H, W, K, psi.device)
    need = search_workspace(N, H, W, V, K) + N * H * W * 8
    ws = alloc_workspace(need, psi.device)
    res = _Result(*[ctypes.c_void_p(out[k].data_ptr()) for k in
                    ("vel_idx", "n_obs", "psi", "phi", "nu", "alpha")])
    rc = lib().kbmod_search_split(_dev(psi, torch.float32, "psi"), _dev(phi, torch.float32, "phi"),
                                  times.ctypes.data_as(ctypes.c_void_p), N, H, W,
                                  vel.ctypes.data_as(ctypes.c_void_p), V, int(K), int(min_obs),
                                  ctypes.byref(res), _dev(ws, torch.uint8, "workspace"),
                                  ctypes.c_size_t(ws.numel()), _stream())
    _check(rc, "kbmod_search_split")
    return out


def eval_trajectories(psiphi: torch.Tensor, times, x0y0: torch.Tensor, vxvy: torch.Tensor,
                      want_pixels: bool = True):
    """kbmod_eval_trajectories (test hook) -> Psi, Phi, n_obs, ixiy (or None)."""
    N, H, W, _ = psiphi.shape
    times = _host(times, np.float64)
    M = x0y0.shape[0]
    dev = psiphi.device
    Psi = torch.empty(M, dtype=torch.float32, device=dev)
    Phi = torch.empty(M, dtype=torch.float32, device=dev)
    nobs = torch.empty(M, dtype=torch.int32, device=dev)
    ixiy = torch.empty((M, N, 2), dtype=torch.int32, device=dev) if want_pixels else None
    rc = lib().kbmod_eval_trajectories(_dev(psiphi, torch.float32, "psiphi"),
                                       times.ctypes.data_as(ctypes.c_void_p), N, H, W,
                                       _dev(x0y0, torch.int32, "x0y0"),
                                       _dev(vxvy, torch.float32, "vxvy"), M,
                                       _dev(Psi, torch.float32, "Psi"), _dev(Phi, torch.float32, "Phi"),
                                       _dev(nobs, torch.int32, "n_obs"),
                                       _dev(ixiy, torch.int32, "ixiy"), _stream())
    _check(rc, "kbmod_eval_trajectories")
    return Psi, Phi, nobs, ixiy


# ----------------------------------------------------------------------------- rows around the search
_CAND_INT, _CAND_FLT = ("x", "y", "vel_idx", "n_obs"), ("psi", "phi", "nu", "alpha")


def search_threshold(psiphi: torch.Tensor, times, vel_grid, min_obs: int, nu_min: float, capacity: int,
                     y_begin: int = 0, y_end: Optional[int] = None, kernel: Optional[int] = None,
                     tile_group_w: int = 0, workspace: Optional[torch.Tensor] = None):
    """kbmod_search_threshold -> (count tensor [1] uint64-as-int64 on the device, dict of device arrays
    [capacity]: x, y, vel_idx, n_obs, psi, phi, nu, alpha).  The first min(count, capacity) entries
    are valid, in unspecified order."""
    N, H, W, two = psiphi.shape
    if two != 2:
        raise KbmodError("psiphi must be [N,H,W,2]")
    times = _host(times, np.float64)
    vel = _host(vel_grid, np.float32)
    if times.shape != (N,) or vel.ndim != 2 or vel.shape[1] != 2:
        raise KbmodError("times must be [N], vel_grid [V,2]")
    V = vel.shape[0]
    y_end = H if y_end is None else int(y_end)
    dev = psiphi.device
    out = {k: torch.empty(max(1, int(capacity)), dtype=torch.int32, device=dev) for k in _CAND_INT}
    out.update({k: torch.empty(max(1, int(capacity)), dtype=torch.float32, device=dev) for k in _CAND_FLT})
    count = torch.zeros(1, dtype=torch.int64, device=dev)
    if workspace is None:
        workspace = alloc_workspace(search_workspace(N, H, W, V, 8), dev)
    cand = _Candidates(*[ctypes.c_void_p(out[k].data_ptr()) for k in _CAND_INT + _CAND_FLT])
    opt = _options(kernel, tile_group_w)
    rc = lib().kbmod_search_threshold(_dev(psiphi, torch.float32, "psiphi"), times.ctypes.data_as(ctypes.c_void_p),
                                      N, H, W, vel.ctypes.data_as(ctypes.c_void_p), V, int(min_obs),
                                      ctypes.c_float(nu_min), int(y_begin), y_end, ctypes.byref(cand),
                                      ctypes.c_longlong(int(capacity)), ctypes.c_void_p(count.data_ptr()),
                                      _dev(workspace, torch.uint8, "workspace"), ctypes.c_size_t(workspace.numel()),
                                      ctypes.byref(opt), _stream())
    _check(rc, "kbmod_search_threshold")
    return count, out


def filter_candidates(psiphi: torch.Tensor, times, x0y0: torch.Tensor, vxvy: torch.Tensor,
                      sigma_reject: float = 5.0, process_var: float = 0.0) -> Dict[str, torch.Tensor]:
    """kbmod_filter_candidates -> dict: psi, phi, nu, alpha [M] f32, n_obs [M] i32, keep [M] i64 (the
    uint64 bit mask), kalman [M,2] f32."""
    N, H, W, _ = psiphi.shape
    times = _host(times, np.float64)
    M = int(x0y0.shape[0])
    dev = psiphi.device
    out = {k: torch.empty(M, dtype=torch.float32, device=dev) for k in ("psi", "phi", "nu", "alpha")}
    out["n_obs"] = torch.empty(M, dtype=torch.int32, device=dev)
    out["keep"] = torch.empty(M, dtype=torch.int64, device=dev)
    out["kalman"] = torch.empty((M, 2), dtype=torch.float32, device=dev)
    if tuple(x0y0.shape) != (M, 2) or tuple(vxvy.shape) != (M, 2) or times.shape != (N,):
        raise KbmodError("x0y0, vxvy must be [M,2], times [N]")
    rc = lib().kbmod_filter_candidates(_dev(psiphi, torch.float32, "psiphi"), times.ctypes.data_as(ctypes.c_void_p),
                                       N, H, W, _dev(x0y0, torch.int32, "x0y0"), _dev(vxvy, torch.float32, "vxvy"), M,
                                       ctypes.c_float(sigma_reject), ctypes.c_float(process_var),
                                       *[ctypes.c_void_p(out[k].data_ptr()) for k in
                                         ("psi", "phi", "n_obs", "nu", "alpha", "keep", "kalman")], _stream())
    _check(rc, "kbmod_filter_candidates")
    return out


def coadd_stamps(sci: torch.Tensor, mask: Optional[torch.Tensor], times, x0y0: torch.Tensor, vxvy: torch.Tensor,
                 keep: Optional[torch.Tensor] = None, R: int = 10):
    """kbmod_coadd_stamps -> stamps [M,2R+1,2R+1] f32, moments [M,6] f32 (m00, cx, cy, mu20, mu02, mu11)."""
    N, H, W = sci.shape
    times = _host(times, np.float64)
    M = int(x0y0.shape[0])
    S = 2 * int(R) + 1
    if tuple(x0y0.shape) != (M, 2) or tuple(vxvy.shape) != (M, 2) or times.shape != (N,):
        raise KbmodError("x0y0, vxvy must be [M,2], times [N]")
    if (mask is not None and mask.shape != sci.shape) or (keep is not None and tuple(keep.shape) != (M,)):
        raise KbmodError("mask must match sci, keep must be [M]")
    stamps = torch.empty((M, S, S), dtype=torch.float32, device=sci.device)
    moments = torch.empty((M, 6), dtype=torch.float32, device=sci.device)
    rc = lib().kbmod_coadd_stamps(_dev(sci, torch.float32, "sci"), _dev(mask, torch.uint8, "mask"),
                                  times.ctypes.data_as(ctypes.c_void_p), N, H, W, _dev(x0y0, torch.int32, "x0y0"),
                                  _dev(vxvy, torch.float32, "vxvy"), _dev(keep, torch.int64, "keep"), M, int(R),
                                  ctypes.c_void_p(stamps.data_ptr()), ctypes.c_void_p(moments.data_ptr()), _stream())
    _check(rc, "kbmod_coadd_stamps")
    return stamps, moments


def build_mask(sci: torch.Tensor, var: torch.Tensor, mask_in: Optional[torch.Tensor] = None, sigma_thr: float = 5.0,
               grow: int = 2, min_images: int = 2, bright_counts: float = 120.0) -> torch.Tensor:
    """kbmod_build_mask -> mask [N,H,W] u8."""
    N, H, W = sci.shape
    if var.shape != sci.shape or (mask_in is not None and mask_in.shape != sci.shape):
        raise KbmodError("sci, var, mask_in shapes differ")
    out = torch.empty((N, H, W), dtype=torch.uint8, device=sci.device)
    rc = lib().kbmod_build_mask(_dev(sci, torch.float32, "sci"), _dev(var, torch.float32, "var"),
                                _dev(mask_in, torch.uint8, "mask_in"), N, H, W, ctypes.c_float(sigma_thr), int(grow),
                                int(min_images), ctypes.c_float(bright_counts), ctypes.c_void_p(out.data_ptr()), _stream())
    _check(rc, "kbmod_build_mask")
    return out


def cluster_candidates(x0y0: torch.Tensor, vxvy: torch.Tensor, nu: torch.Tensor, eps_xy: float = 2.0,
                       eps_v: float = 4.0, min_samples: int = 1):
    """kbmod_cluster_candidates -> label [M] i32 (-1 = noise), rep [M] u8.  Synchronises the stream."""
    M = int(x0y0.shape[0])
    if tuple(x0y0.shape) != (M, 2) or tuple(vxvy.shape) != (M, 2) or tuple(nu.shape) != (M,):
        raise KbmodError("x0y0, vxvy must be [M,2], nu [M]")
    dev = x0y0.device
    label = torch.empty(M, dtype=torch.int32, device=dev)
    rep = torch.empty(M, dtype=torch.uint8, device=dev)
    ws = alloc_workspace(lib().kbmod_cluster_workspace(M), dev)
    rc = lib().kbmod_cluster_candidates(_dev(x0y0, torch.int32, "x0y0"), _dev(vxvy, torch.float32, "vxvy"),
                                        _dev(nu, torch.float32, "nu"), M, ctypes.c_float(eps_xy), ctypes.c_float(eps_v),
                                        int(min_samples), ctypes.c_void_p(label.data_ptr()), ctypes.c_void_p(rep.data_ptr()),
                                        _dev(ws, torch.uint8, "workspace"), ctypes.c_size_t(ws.numel()), _stream())
    _check(rc, "kbmod_cluster_candidates")
    return label, rep
