"""GPU parity: the CUDA path (through the C ABI) against the CPU oracle on the same seeded inputs.

Bars (BASELINE.json north_star):
  psi/phi images : |gpu - oracle| <= 1e-5 * sum|terms| + 1e-7, invalid markers identical
  search         : vel_idx, n_obs and sampled pixels bit-exact; Psi/Phi/nu/alpha bit-exact against
                   the oracle's f32seq mode (same rounding order), and within rel 1e-5 (abs 1e-4
                   when |nu| < 1) of its f64 mode, top-K sets equal up to near-tie swaps.
"""
import math
import os

import numpy as np
import pytest
import torch

from paper_1901_02492_b200 import synth

# KBMOD_GPU_TESTS_EMULATED=1: run this file's LOGIC against the SIMT-emulated library on CPU tensors
EMULATED = os.environ.get("KBMOD_GPU_TESTS_EMULATED") == "1"
pytestmark = pytest.mark.gpu

# 1 = direct gather, 0 = automatic (the tiled kernel where the shape fits), 3 = TMA-staged kernel.
# The staged kernel has not yet been validated on hardware: it is only
# exercised when KBMOD_TEST_STAGED=1, so that an untested kernel cannot take the suite down.
KERNELS = [1, 0] + ([3] if os.environ.get("KBMOD_TEST_STAGED") == "1" else [])


@pytest.fixture(scope="module")
def kb():
    if EMULATED:                     # test-logic check on a machine without a GPU (tests/emulated_binding.py)
        from tests import emulated_binding as binding
    else:
        from paper_1901_02492_b200 import binding
        if not torch.cuda.is_available():
            pytest.fail("GPU tests need a CUDA device (no CPU fallback exists)")
    binding.lib()
    yield binding
    binding.set_search_kernel(0)


def _cuda(a):
    t = torch.from_numpy(np.ascontiguousarray(a))
    return t if EMULATED else t.cuda()


def _np(res):
    return {k: v.cpu().numpy() for k, v in res.items()}


def assert_psiphi_close(gpu, ref, pabs):
    gn, rn = np.isnan(gpu[..., 0]), np.isnan(ref[..., 0])
    assert (gn == rn).all(), "invalid markers differ"
    assert (gpu[..., 1][rn] == 0).all()
    ok = ~rn
    tol_psi = 1e-5 * pabs[ok] + 1e-7
    assert (np.abs(gpu[..., 0][ok] - ref[..., 0][ok]) <= tol_psi).all()
    tol_phi = 1e-5 * ref[..., 1][ok] + 1e-7
    assert (np.abs(gpu[..., 1][ok] - ref[..., 1][ok]) <= tol_phi).all()


def assert_search_exact(gpu, ref):
    """Against the oracle's f32seq mode: everything identical, bit for bit."""
    for k in ("vel_idx", "n_obs"):
        assert (gpu[k] == ref[k]).all(), k
    for k in ("psi", "phi", "nu", "alpha"):
        assert (gpu[k].view(np.int32) == ref[k].view(np.int32)).all() or \
            ((gpu[k] == ref[k]) | (np.isnan(gpu[k]) & np.isnan(ref[k]))).all(), k


def assert_search_close_f64(gpu, ref):
    """Against the oracle's f64 mode: values within tolerance; slots may swap only between
    candidates whose nu differ by less than the tolerance."""
    def tol(nu):
        return np.where(np.abs(nu) < 1.0, 1e-4, 1e-5 * np.abs(nu))
    real_g, real_r = gpu["vel_idx"] >= 0, ref["vel_idx"] >= 0
    assert (real_g == real_r).all()
    nu_g = np.where(real_g, gpu["nu"], 0.0)
    nu_r = np.where(real_r, ref["nu"], 0.0)
    assert (np.abs(nu_g - nu_r) <= tol(nu_r)).all()          # sorted lists agree slot by slot
    same = gpu["vel_idx"] == ref["vel_idx"]
    for k in ("psi", "phi", "alpha"):
        a, b = gpu[k][same & real_g], ref[k][same & real_g]
        assert (np.abs(a - b) <= 1e-5 * np.abs(b) + 1e-4 * (np.abs(b) < 1)).all(), k
    assert (gpu["n_obs"][same] == ref["n_obs"][same]).all()
    # a differing slot must be a near tie: its velocity appears elsewhere in the other list
    # (or sits at the K boundary) with nu within tolerance
    for (y, x, k) in np.argwhere(~same):
        j = gpu["vel_idx"][y, x, k]
        pos = np.flatnonzero(ref["vel_idx"][y, x] == j)
        if len(pos):
            assert abs(ref["nu"][y, x, pos[0]] - gpu["nu"][y, x, k]) <= 2 * tol(ref["nu"][y, x, k])
        else:
            assert abs(ref["nu"][y, x, -1] - gpu["nu"][y, x, k]) <= 2 * tol(ref["nu"][y, x, -1])


# ------------------------------------------------------------------------------ psi/phi
@pytest.mark.parametrize("k,over", [
    (1, {}),
    (2, dict(N=3, H=150, W=210)),                     # several tiles + ragged tail, P=19
    (3, dict(N=2, H=97, W=131, n_sources=5)),         # P=21, variance gradient
    (4, dict(N=2, H=120, W=136, n_sources=5)),        # elliptical (non rank-1) PSF, P=27, 10% mask
])
def test_psi_phi_matches_oracle(kb, orc, k, over):
    st = synth.make_stack(synth.config(k, **over))
    ref, pabs = orc.make_psi_phi(st.sci, st.var, st.mask, st.psf, want_abs=True)
    gpu = kb.make_psi_phi(_cuda(st.sci), _cuda(st.var), _cuda(st.mask), st.psf).cpu().numpy()
    assert_psiphi_close(gpu, ref, pabs)


def test_psi_phi_edge_cases(kb, orc):
    rng = np.random.default_rng(0)
    # 1x1 PSF, tiny image, no mask pointer, bad numerics
    sci = rng.standard_normal((2, 5, 7)).astype(np.float32)
    var = rng.uniform(1, 2, (2, 5, 7)).astype(np.float32)
    sci[0, 1, 1] = np.nan
    sci[1, 2, 3] = np.inf
    var[0, 3, 3] = 0.0
    var[1, 0, 0] = -1.0
    var[1, 4, 6] = np.inf
    for P in (1, 3, 31):
        psf = rng.uniform(0.0, 1.0, (2, P, P)).astype(np.float32)
        psf[:, P // 2, P // 2] = 1.0
        ref, pabs = orc.make_psi_phi(sci, var, None, psf, want_abs=True)
        gpu = kb.make_psi_phi(_cuda(sci), _cuda(var), None, psf).cpu().numpy()
        assert_psiphi_close(gpu, ref, pabs)
    # asymmetric kernel: correlation, not convolution
    psf = np.zeros((2, 5, 5), np.float32)
    psf[:, 3, 4] = 1.0
    psf[:, 2, 2] = 0.5
    ref, pabs = orc.make_psi_phi(sci, var, None, psf, want_abs=True)
    gpu = kb.make_psi_phi(_cuda(sci), _cuda(var), None, psf).cpu().numpy()
    assert_psiphi_close(gpu, ref, pabs)
    # fully masked image
    mask = np.ones((2, 5, 7), np.uint8)
    gpu = kb.make_psi_phi(_cuda(sci), _cuda(var), _cuda(mask), psf).cpu().numpy()
    assert np.isnan(gpu[..., 0]).all() and (gpu[..., 1] == 0).all()


# ------------------------------------------------------------------------------ search
@pytest.mark.parametrize("which", KERNELS)
def test_search_config1_end_to_end(kb, orc, which):
    kb.set_search_kernel(which)
    cfg = synth.config(1)
    st = synth.make_stack(cfg)
    pp_ref = orc.make_psi_phi(st.sci, st.var, st.mask, st.psf)
    # (a) both searches fed the oracle's psi/phi: exact
    gpu = _np(kb.search(_cuda(pp_ref), st.times, st.vel_grid, cfg.K, cfg.min_obs))
    assert_search_exact(gpu, orc.search(pp_ref, st.times, st.vel_grid, cfg.K, cfg.min_obs))
    assert_search_close_f64(gpu, orc.search(pp_ref, st.times, st.vel_grid, cfg.K, cfg.min_obs,
                                            mode=orc.MODE_F64))
    # (b) end to end, each side on its own psi/phi: the injected source is recovered
    pp_gpu = kb.make_psi_phi(_cuda(st.sci), _cuda(st.var), _cuda(st.mask), st.psf)
    e2e = _np(kb.search(pp_gpu, st.times, st.vel_grid, cfg.K, cfg.min_obs))
    y, x = np.unravel_index(np.argmax(e2e["nu"][..., 0]), e2e["nu"].shape[:2])
    assert (x, y) == (20, 30) and e2e["vel_idx"][y, x, 0] == 19
    ref = orc.search(pp_ref, st.times, st.vel_grid, cfg.K, cfg.min_obs)
    np.testing.assert_allclose(e2e["nu"][y, x], ref["nu"][y, x], rtol=1e-5)


@pytest.mark.parametrize("which", KERNELS)
@pytest.mark.parametrize("k,over", [
    (2, dict(N=8, H=75, W=203)),
    (3, dict(N=15, H=70, W=133, n_sources=4)),
    (4, dict(N=12, H=66, W=140, n_sources=4, n_angles=16, n_speeds=8)),
    (5, dict(N=20, H=40, W=97, n_angles=8, n_speeds=8)),
])
def test_search_crops_match_oracle_exactly(kb, orc, which, k, over):
    """Crops of configs 2-5 (full time base, full velocity range => most trajectories leave the
    image: exercises edges and n_obs < min_obs heavily)."""
    kb.set_search_kernel(which)
    cfg = synth.config(k, **over)
    st = synth.make_stack(cfg)
    pp = orc.make_psi_phi(st.sci, st.var, st.mask, st.psf)
    gpu = _np(kb.search(_cuda(pp), st.times, st.vel_grid, cfg.K, cfg.min_obs))
    assert_search_exact(gpu, orc.search(pp, st.times, st.vel_grid, cfg.K, cfg.min_obs))


@pytest.mark.parametrize("which", KERNELS)
def test_search_slow_velocities_interior(kb, orc, which):
    """Velocities scaled so trajectories stay inside a small image: full n_obs, real top-K."""
    kb.set_search_kernel(which)
    pp = synth.random_psiphi(9, 150, 260, seed=21, invalid_frac=0.03)
    times = np.array([0, .05, .1, .15, 1, 1.05, 1.1, 2.0, 2.05])
    vel = synth.velocity_grid(12, 10, -math.pi / 3, math.pi / 3, 3.0, 40.0)
    for K, mo in ((8, 5), (16, 9), (3, 1), (32, 2)):
        gpu = _np(kb.search(_cuda(pp), times, vel, K, mo))
        assert_search_exact(gpu, orc.search(pp, times, vel, K, mo))
    assert_search_close_f64(gpu, orc.search(pp, times, vel, 32, 2, mode=orc.MODE_F64))


@pytest.mark.parametrize("which", KERNELS)
def test_search_edge_cases(kb, orc, which):
    kb.set_search_kernel(which)
    rng = np.random.default_rng(4)
    # N = 1, V = 1, K > V (sentinels), 1-pixel-high image
    pp = synth.random_psiphi(1, 1, 33, seed=1, invalid_frac=0.2)
    gpu = _np(kb.search(_cuda(pp), [3.0], np.zeros((1, 2), np.float32), 4, 1))
    assert_search_exact(gpu, orc.search(pp, [3.0], np.zeros((1, 2), np.float32), 4, 1))
    # all-NaN stack: nothing eligible anywhere
    pp = synth.random_psiphi(3, 20, 40, seed=2, invalid_frac=1.1)
    vel = synth.velocity_grid(3, 3, -1, 1, 1, 5)
    gpu = _np(kb.search(_cuda(pp), [0, 1, 2], vel, 5, 1))
    assert (gpu["vel_idx"] == -1).all() and np.isneginf(gpu["nu"]).all()
    assert (gpu["n_obs"] == 0).all() and (gpu["psi"] == 0).all() and (gpu["alpha"] == 0).all()
    # duplicated velocities (ties -> smaller index first), unsorted times, negative time steps
    pp = synth.random_psiphi(5, 37, 70, seed=3, invalid_frac=0.1)
    vel = synth.velocity_grid(4, 4, -2, 2, 2, 12)
    vel = np.concatenate([vel, vel[3:9], vel[:2]])
    times = np.array([5.0, 4.5, 6.0, 5.25, 7.0])
    gpu = _np(kb.search(_cuda(pp), times, vel, 8, 2))
    assert_search_exact(gpu, orc.search(pp, times, vel, 8, 2))
    # min_obs = N: only fully observed trajectories
    gpu = _np(kb.search(_cuda(pp), times, vel, 8, 5))
    assert_search_exact(gpu, orc.search(pp, times, vel, 8, 5))
    # phi == 0 with valid psi (allowed by the contract): counted, eligible only if Phi > 0
    pp2 = pp.copy()
    pp2[..., 1] = np.where(rng.random(pp2.shape[:-1]) < 0.5, 0.0, pp2[..., 1])
    gpu = _np(kb.search(_cuda(pp2), times, vel, 8, 2))
    assert_search_exact(gpu, orc.search(pp2, times, vel, 8, 2))


@pytest.mark.parametrize("which", KERNELS)
def test_search_half_integer_and_near_tie_positions(kb, orc, which):
    """P5 through the search: velocities whose v*dt are exact halves or within 2^-10 of one
    (the pairs for which a per-velocity integer offset is NOT the definition)."""
    kb.set_search_kernel(which)
    H, W = 40, 4096
    pp = np.zeros((3, H, W, 2), np.float32)
    pp[1:, ..., 0] = (np.arange(H)[:, None] * W + np.arange(W)[None, :]).astype(np.float32)[None]
    pp[..., 1] = 1.0
    times = np.array([0.0, 0.5, 1.0])
    vel = np.array([[3.0, 1.0], [-3.0, -1.0], [1.0, 3.0], [10.49999, 0.0], [20.99998, 0.5],
                    [0.49999997, 0.49999997], [0.99999994, -0.99999994], [7.0, 7.0],
                    [-0.5, 0.0], [2047.5, 0.0], [4095.0, 1.0], [10.5, 10.5]], np.float32)
    gpu = _np(kb.search(_cuda(pp), times, vel, 12, 1))
    assert_search_exact(gpu, orc.search(pp, times, vel, 12, 1))


def test_eval_trajectories_pixels_bit_exact(kb, orc):
    rng = np.random.default_rng(9)
    pp = synth.random_psiphi(7, 90, 4096, seed=5, invalid_frac=0.05)
    times = np.sort(rng.uniform(0, 3.2, 7))
    M = 5000
    x0y0 = np.stack([rng.integers(0, 4096, M), rng.integers(0, 90, M)], 1).astype(np.int32)
    vxvy = rng.uniform(-600, 600, (M, 2)).astype(np.float32)
    vxvy[:200] = np.round(vxvy[:200] * 2) / 2            # exact halves at dt multiples
    Psi, Phi, nobs, ixiy = [t.cpu().numpy() for t in
                            kb.eval_trajectories(_cuda(pp), times, _cuda(x0y0), _cuda(vxvy))]
    rPsi, rPhi, rn, rix = orc.eval_trajectories(pp, times, x0y0, vxvy)
    assert (ixiy == rix).all() and (nobs == rn).all()
    assert (Psi == rPsi).all() and (Phi == rPhi).all()


def test_search_split_entry_point(kb, orc):
    pp = synth.random_psiphi(4, 30, 50, seed=6)
    vel = synth.velocity_grid(3, 3, -1, 1, 2, 9)
    times = [0.0, 0.3, 0.6, 1.4]
    g = _np(kb.search_split(_cuda(pp[..., 0]), _cuda(pp[..., 1]), times, vel, 4, 2))
    assert_search_exact(g, orc.search(pp, times, vel, 4, 2))


@pytest.mark.parametrize("which", KERNELS)
def test_search_row_bands_concatenate_to_the_full_search(kb, orc, which):
    """kbmod_search_rows ("entirely independent"): disjoint bands of
    start rows of one stack, searched one after the other on this GPU, concatenate to the full
    search bit for bit; the planes hold the band only; a prebuilt kbmod_plan gives the same."""
    kb.set_search_kernel(which)
    cfg = synth.config(2, N=8, H=75, W=203)
    st = synth.make_stack(cfg)
    pp = orc.make_psi_phi(st.sci, st.var, st.mask, st.psf)
    d_pp = _cuda(pp)
    full = _np(kb.search(d_pp, st.times, st.vel_grid, cfg.K, cfg.min_obs))
    assert_search_exact(full, orc.search(pp, st.times, st.vel_grid, cfg.K, cfg.min_obs))
    from paper_1901_02492_b200 import shard
    for world in (2, 3):
        parts = [_np(kb.search(d_pp, st.times, st.vel_grid, cfg.K, cfg.min_obs, y_begin=y0, y_end=y1))
                 for y0, y1 in shard.row_bands(cfg.H, world)]
        cat = {k: np.concatenate([p[k] for p in parts], 0) for k in full}
        assert_search_exact(cat, full)
    plan = kb.Plan(st.times, cfg.N, cfg.H, cfg.W, st.vel_grid, cfg.K)
    for y0, y1 in ((0, cfg.H), (31, 33), (74, 75), (40, 40)):
        band = _np(kb.search(d_pp, None, None, cfg.K, cfg.min_obs, y_begin=y0, y_end=y1, plan=plan))
        assert band["nu"].shape == (y1 - y0, cfg.W, cfg.K)
        assert_search_exact(band, {k: v[y0:y1] for k, v in full.items()})
    plan.close()


def test_errors_are_loud(kb):
    pp = _cuda(synth.random_psiphi(2, 8, 8, seed=1))
    with pytest.raises(kb.KbmodError):
        kb.search(pp, [0.0, 1.0], np.zeros((1, 2), np.float32), 40, 1)        # K > 32
    with pytest.raises(kb.KbmodError):
        kb.search(pp, [0.0, np.nan], np.zeros((1, 2), np.float32), 2, 1)      # bad time
    if not EMULATED:
        with pytest.raises(kb.KbmodError):
            kb.search(pp.cpu(), [0.0, 1.0], np.zeros((1, 2), np.float32), 2, 1)   # host tensor


# ------------------------------------------------------------------------------ added after the last GPU run
# The tests below were written after GPU access closed in round 1: they sit at
# the end of the file so that every test that has already passed on hardware reports first.
@pytest.mark.parametrize("which", KERNELS)
def test_search_maximum_image_count(kb, orc, which):
    """N = KBMOD_MAX_IMAGES = 64 (and N = 40, the largest stack of BASELINE.json configs[4])."""
    kb.set_search_kernel(which)
    rng = np.random.default_rng(64)
    for N, mo in ((64, 20), (40, 20)):
        pp = synth.random_psiphi(N, 40, 70, seed=N, invalid_frac=0.05)
        times = np.sort(rng.uniform(0.0, 5.0, N))
        vel = synth.velocity_grid(6, 4, -math.pi / 2, math.pi / 2, 1.0, 9.0)
        gpu = _np(kb.search(_cuda(pp), times, vel, 8, mo))
        assert_search_exact(gpu, orc.search(pp, times, vel, 8, mo))
    with pytest.raises(kb.KbmodError):                                        # N = 65: beyond the limit
        kb.search(_cuda(synth.random_psiphi(65, 4, 4, seed=1)), np.arange(65.0), vel, 2, 1)


def test_search_host_entry_point(kb, orc):
    """kbmod_search_host (HOST buffers in, HOST planes out) equals the two device-pointer calls."""
    cfg = synth.config(2, N=8, H=75, W=203)
    st = synth.make_stack(cfg)
    pin = lambda a: (lambda t: t if EMULATED else t.pin_memory())(torch.from_numpy(np.ascontiguousarray(a)))
    out = {k: torch.empty((cfg.H, cfg.W, cfg.K), dtype=torch.int32 if k in ("vel_idx", "n_obs") else torch.float32)
           for k in ("vel_idx", "n_obs", "psi", "phi", "nu", "alpha")}
    if not EMULATED:
        out = {k: v.pin_memory() for k, v in out.items()}
    ws = kb.alloc_workspace(kb.search_host_workspace(cfg.N, cfg.H, cfg.W, cfg.V, cfg.K), "cpu" if EMULATED else "cuda")
    kb.search_host(pin(st.sci), pin(st.var), pin(st.mask), st.psf, st.times, st.vel_grid, cfg.K, cfg.min_obs, out, ws)
    kb.search_status(ws)                                  # synchronises
    pp = kb.make_psi_phi(_cuda(st.sci), _cuda(st.var), _cuda(st.mask), st.psf)
    ref = _np(kb.search(pp, st.times, st.vel_grid, cfg.K, cfg.min_obs))
    assert_search_exact({k: v.numpy() for k, v in out.items()}, ref)
    # and the oracle agrees on the same psi/phi
    assert_search_exact(ref, orc.search(pp.cpu().numpy(), st.times, st.vel_grid, cfg.K, cfg.min_obs))


# ------------------------------------------------------------------------------ full size
@pytest.mark.parametrize("which", [k for k in KERNELS if k != 1])
def test_search_full_size_config3_sampled_bands(kb, orc, which):
    """BASELINE.json configs[2] at full size, in the launch configuration bench.py times (GPU
    psi/phi feeding the default search kernel): bands of start rows at the image edges, across
    tile boundaries and in the interior are recomputed by the oracle on the same psi/phi and
    must match bit for bit (every start pixel of the band, all K slots)."""
    kb.set_search_kernel(which)
    cfg = synth.config(3)
    st = synth.make_stack(cfg)
    pp = kb.make_psi_phi(_cuda(st.sci), _cuda(st.var), _cuda(st.mask), st.psf)
    res = kb.search(pp, st.times, st.vel_grid, cfg.K, cfg.min_obs)
    pp_host = pp.cpu().numpy()
    del pp
    for y0 in (0, 28, 2044, cfg.H - 8):            # 8-row bands; 28..36 straddles a 30/32-row tile edge
        ref = orc.search(pp_host, st.times, st.vel_grid, cfg.K, cfg.min_obs, y_begin=y0, y_end=y0 + 8)
        gpu = {k: v[y0:y0 + 8].cpu().numpy() for k, v in res.items()}
        assert_search_exact(gpu, ref)
    # the injected sources are there: the best nu of the frame is far above the noise maximum (~6.5)
    best = float(res["nu"][..., 0].max().item())
    assert best > 8.0


# ------------------------------------------------------------------------------ every BASELINE.json config at size
def _full_size_case(kb, orc, cfg, bands):
    """psi/phi + search at full size with the default kernel (the launch configuration bench.py
    times); 8-row bands of start rows are recomputed by the oracle on the same psi/phi and must
    match bit for bit; psi/phi itself is compared with the oracle on the same bands (inputs cropped
    with the PSF halo) at the section 8(c) tolerance."""
    kb.set_search_kernel(0)
    st = synth.make_stack(cfg)
    pp = kb.make_psi_phi(_cuda(st.sci), _cuda(st.var), _cuda(st.mask), st.psf)
    res = kb.search(pp, st.times, st.vel_grid, cfg.K, cfg.min_obs)
    r = (st.psf.shape[-1] - 1) // 2
    for y0 in bands:
        a, b = max(0, y0 - r), min(cfg.H, y0 + 8 + r)
        ref_pp, pabs = orc.make_psi_phi(st.sci[:, a:b], st.var[:, a:b], st.mask[:, a:b], st.psf, want_abs=True)
        # rows whose stencil is cut by the crop (not by the image) are not comparable: keep the band only
        sl = slice(y0 - a, y0 - a + 8)
        assert_psiphi_close(pp[:, y0:y0 + 8].cpu().numpy(), ref_pp[:, sl], pabs[:, sl])
    pp_host = pp.cpu().numpy()
    del pp
    for y0 in bands:
        ref = orc.search(pp_host, st.times, st.vel_grid, cfg.K, cfg.min_obs, y_begin=y0, y_end=y0 + 8)
        gpu = {k: v[y0:y0 + 8].cpu().numpy() for k, v in res.items()}
        assert_search_exact(gpu, ref)
    return res


def test_full_size_config2_ccd_night_pair(kb, orc):
    """BASELINE.json configs[1] whole: 8 x 2048 x 4096, V = 512, K = 8, P = 19."""
    cfg = synth.config(2)
    res = _full_size_case(kb, orc, cfg, (0, 28, 1020, cfg.H - 8))
    assert float(res["nu"][..., 0].max().item()) > 8.0          # the injected sources are there


def test_full_size_config4_stress(kb, orc):
    """BASELINE.json configs[3] whole: 12 x 4096 x 4096, V = 2048, K = 16 (64 x 16 tiles), P = 27
    rotated elliptical PSFs (general 2-D psi/phi path), 10 % static + random masks, irregular times."""
    cfg = synth.config(4)
    _full_size_case(kb, orc, cfg, (0, 12, 2040, cfg.H - 8))


@pytest.mark.parametrize("N,V", [(40, 640), (10, 8192)])
def test_full_size_config5_sweep_corners(kb, orc, N, V):
    """BASELINE.json configs[4], the two far corners of the sweep: the deepest stack (N = 40,
    additive counters, 5.4 GB of psi/phi) and the largest grid (V = 8192, +-pi/2, up to 800 px/day)."""
    na, ns = synth.SWEEP_GRIDS[V]
    cfg = synth.config(5, N=N, n_angles=na, n_speeds=ns)
    _full_size_case(kb, orc, cfg, (0, 2044, cfg.H - 8))
