"""GPU parity of the rows around the search, through the C ABI against the
CPU oracle on the same seeded inputs: N4 threshold-mode search, N1 light-curve filter, N2 coadded
stamps and moments, N3 mask builder, N5 DBSCAN de-duplication.  Bars: every integer / bit-mask / index output bit-exact; every
float bit-exact too (each is a fixed sequence of separately rounded binary32 operations that the
oracle restates).  The device logic of these kernels is checked on the CPU first
(tests/test_post_simt.py, also under AddressSanitizer); this file sorts after tests/test_gpu_parity.py.
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
CAND = ("x", "y", "vel_idx", "n_obs", "psi", "phi", "nu", "alpha")


@pytest.fixture(scope="module")
def kb():
    if EMULATED:                     # test-logic check on a machine without a GPU (tests/emulated_binding.py)
        from tests import emulated_binding as binding
    else:
        from paper_1901_02492_b200 import binding
        if not torch.cuda.is_available():
            pytest.fail("GPU tests need a CUDA device (no CPU fallback exists)")
    binding.lib()
    return binding


def _cuda(a):
    t = torch.from_numpy(np.ascontiguousarray(a))
    return t if EMULATED else t.cuda()


def _bits(a, b):
    return ((a.view(np.int32) == b.view(np.int32)) | (a == b)).all() if a.dtype == np.float32 else (a == b).all()


def _sorted(c):
    o = np.lexsort((c["vel_idx"], c["x"], c["y"]))
    return {k: v[o] for k, v in c.items()}


# queued-kernel variant: opt-in like the rest of kernel 4 (tests/test_zz_gpu_queued_kernel.py)
THRESH_KERNELS = [0] + ([4] if os.environ.get("KBMOD_TEST_QUEUED") == "1" else [])


@pytest.mark.parametrize("kernel", THRESH_KERNELS)
def test_threshold_search_matches_oracle_set(kb, orc, kernel):
    cfg = synth.config(1)
    st = synth.make_stack(cfg)
    pp = orc.make_psi_phi(st.sci, st.var, st.mask, st.psf)
    cases = [(pp, st.times, st.vel_grid, cfg.min_obs, 4.0, 0, cfg.H)]
    pp2 = synth.random_psiphi(9, 150, 260, seed=21, invalid_frac=0.03)
    t2 = np.array([0, .05, .1, .15, 1, 1.05, 1.1, 2.0, 2.05])
    v2 = synth.velocity_grid(12, 10, -math.pi / 3, math.pi / 3, 3.0, 40.0)
    cases += [(pp2, t2, v2, 5, 2.0, 0, 150), (pp2, t2, v2, 9, 1.0, 40, 111)]
    for pp_, t_, v_, mo, thr, y0, y1 in cases:
        n_ref, ref = orc.search_threshold(pp_, t_, v_, mo, thr, y0, y1)
        count, got = kb.search_threshold(_cuda(pp_), t_, v_, mo, thr, n_ref + 100, y0, y1, kernel=kernel)
        n = int(count.item())
        assert n == n_ref and n > 0
        got = _sorted({k: v[:n].cpu().numpy() for k, v in got.items()})
        ref = _sorted(ref)
        for k in CAND:
            assert _bits(got[k], ref[k]), k
        count, _ = kb.search_threshold(_cuda(pp_), t_, v_, mo, thr, 5, y0, y1, kernel=kernel)     # overflow: count exact
        assert int(count.item()) == n_ref
    # the injected source of config 1 is the only thing above 20 sigma
    pp_gpu = kb.make_psi_phi(_cuda(st.sci), _cuda(st.var), _cuda(st.mask), st.psf)
    count, got = kb.search_threshold(pp_gpu, st.times, st.vel_grid, cfg.min_obs, 20.0, 1000, kernel=kernel)
    n = int(count.item())
    assert 1 <= n < 200
    best = int(torch.argmax(got["nu"][:n]).item())
    assert abs(int(got["x"][best]) - 20) <= 1 and abs(int(got["y"][best]) - 30) <= 1


def test_filter_candidates_matches_oracle(kb, orc):
    rng = np.random.default_rng(17)
    for N, frac, q, sigma in ((15, 0.1, 0.0, 5.0), (15, 0.1, 3.5, 3.0), (64, 0.3, 0.25, 2.0), (1, 0.0, 0.0, 5.0)):
        H, W, M = 90, 130, 20000
        pp = synth.random_psiphi(N, H, W, seed=100 + N, invalid_frac=frac)
        pp[..., 1] = np.where(rng.random((N, H, W)) < 0.02, 0.0, pp[..., 1])
        pp[..., 0] = np.where(rng.random((N, H, W)) < 0.05, pp[..., 0] * 60.0, pp[..., 0])
        times = np.sort(rng.uniform(0, 3.0, N))
        x0y0 = np.stack([rng.integers(0, W, M), rng.integers(0, H, M)], 1).astype(np.int32)
        vxvy = rng.uniform(-12, 12, (M, 2)).astype(np.float32)
        ref = orc.filter_candidates(pp, times, x0y0, vxvy, sigma, q)
        got = {k: v.cpu().numpy() for k, v in
               kb.filter_candidates(_cuda(pp), times, _cuda(x0y0), _cuda(vxvy), sigma, q).items()}
        assert (got["keep"].view(np.uint64) == ref["keep"]).all() and (got["n_obs"] == ref["n_obs"]).all()
        for k in ("psi", "phi", "nu", "alpha", "kalman"):
            assert _bits(got[k], ref[k]), (k, N)


def test_search_then_filter_removes_an_interloper(kb, orc):
    """The paper's Fig.3 case end to end on the GPU: top-K search, then the light-curve filter on
    the winners; a trajectory that is bright only because ONE image has a bright pixel on it loses
    that observation and its likelihood collapses, while the real source keeps all of its."""
    cfg = synth.config(1)
    st = synth.make_stack(cfg)
    st.sci[3, 50, 10] += 4000.0                                      # an interloper in one image
    pp = kb.make_psi_phi(_cuda(st.sci), _cuda(st.var), _cuda(st.mask), st.psf)
    res = kb.search(pp, st.times, st.vel_grid, 1, 3)
    nu = res["nu"][..., 0]
    flat = torch.topk(nu.flatten(), 200).indices
    ys, xs = (flat // cfg.W).int(), (flat % cfg.W).int()
    x0y0 = torch.stack([xs, ys], 1).contiguous()
    vel = _cuda(st.vel_grid)[res["vel_idx"][..., 0].flatten()[flat].long()].contiguous()
    out = kb.filter_candidates(pp, st.times, x0y0, vel)
    ref = orc.filter_candidates(pp.cpu().numpy(), st.times, x0y0.cpu().numpy(), vel.cpu().numpy())
    assert (out["keep"].cpu().numpy().view(np.uint64) == ref["keep"]).all()
    before, after = nu.flatten()[flat].cpu().numpy(), out["nu"].cpu().numpy()
    src = (xs.cpu().numpy() == 20) & (ys.cpu().numpy() == 30)
    assert src.any() and (after[src] == before[src]).all() and (out["n_obs"].cpu().numpy()[src] == 5).all()
    dropped = out["n_obs"].cpu().numpy() < res["n_obs"][..., 0].flatten()[flat].cpu().numpy()
    assert dropped.any() and (after[dropped] < 0.5 * before[dropped]).any()


def test_coadd_stamps_and_moments_match_oracle(kb, orc):
    rng = np.random.default_rng(23)
    N, H, W = 9, 120, 160
    sci = rng.normal(0, 10, (N, H, W)).astype(np.float32)
    sci[:, 50:55, 70:75] += 300.0
    sci[2, 52, 71] = np.nan
    mask = (rng.random((N, H, W)) < 0.05).astype(np.uint8)
    times = np.sort(rng.uniform(0, 2.0, N))
    M = 3000
    x0y0 = np.stack([rng.integers(0, W, M), rng.integers(0, H, M)], 1).astype(np.int32)
    x0y0[:3] = [[0, 0], [W - 1, H - 1], [72, 52]]
    vxvy = rng.uniform(-8, 8, (M, 2)).astype(np.float32)
    vxvy[2] = 0.0
    keep = rng.integers(0, 1 << N, M).astype(np.int64)
    keep[2] = (1 << N) - 1
    for R, msk, kp in ((10, mask, keep), (3, None, None), (0, mask, None), (15, None, keep)):
        st_ref, mo_ref = orc.coadd_stamps(sci, msk, times, x0y0, vxvy, None if kp is None else kp.astype(np.uint64), R)
        st, mo = kb.coadd_stamps(_cuda(sci), None if msk is None else _cuda(msk), times, _cuda(x0y0), _cuda(vxvy),
                                 None if kp is None else _cuda(kp), R)
        assert _bits(st.cpu().numpy(), st_ref) and _bits(mo.cpu().numpy(), mo_ref), R


def test_build_mask_matches_oracle_and_feeds_psi_phi(kb, orc):
    rng = np.random.default_rng(29)
    for (N, H, W, grow, mi) in ((4, 150, 210, 2, 2), (3, 33, 31, 0, 1), (6, 97, 131, 8, 3)):
        var = rng.uniform(80, 150, (N, H, W)).astype(np.float32)
        sci = (rng.normal(0, 1, (N, H, W)) * np.sqrt(var) * 2.2).astype(np.float32)
        for _ in range(12):
            y, x = rng.integers(0, H), rng.integers(0, W)
            sci[:, y, x] += 500.0
        sci[0, 0, 0] = np.nan
        var[0, H - 1, W - 1] = -1.0
        mask_in = (rng.random((N, H, W)) < 0.01).astype(np.uint8)
        for m_in in (mask_in, None):
            want = orc.build_mask(sci, var, m_in, 5.0, grow, mi, 120.0)
            got = kb.build_mask(_cuda(sci), _cuda(var), None if m_in is None else _cuda(m_in), 5.0, grow, mi, 120.0)
            assert (got.cpu().numpy() == want).all()
    # the built mask goes straight into kbmod_make_psi_phi (device to device)
    psf = synth.gaussian_psf_kernels([1.2] * N, [1.2] * N, [0.0] * N, 7)
    pp = kb.make_psi_phi(_cuda(sci), _cuda(var), got, psf).cpu().numpy()
    assert (np.isnan(pp[..., 0]) == (want != 0) | ~np.isfinite(sci) | ~(var > 0)).all()


def test_cluster_candidates_matches_oracle(kb, orc):
    """N5 on the device: canonical DBSCAN labels and representatives equal the oracle's, and the
    whole chain search -> threshold list -> de-duplication collapses the near-duplicates around the
    injected source of config 1 and keeps its brightest trajectory."""
    rng = np.random.default_rng(61)
    centres = np.stack([rng.integers(0, 300, 30), rng.integers(0, 300, 30), rng.integers(-30, 30, 30) * 4,
                        rng.integers(-30, 30, 30) * 4], 1)
    pts = np.concatenate([centres[rng.integers(0, 30, 3000)] +
                          np.stack([rng.integers(-2, 3, 3000), rng.integers(-2, 3, 3000), rng.integers(-2, 3, 3000) * 2,
                                    rng.integers(-2, 3, 3000) * 2], 1),
                          np.stack([rng.integers(0, 300, 200), rng.integers(0, 300, 200), rng.integers(-120, 120, 200),
                                    rng.integers(-120, 120, 200)], 1),
                          np.stack([np.arange(900)[::-1] * 2 + 1000, np.zeros(900, int), np.zeros(900, int),
                                    np.zeros(900, int)], 1)])
    x0y0, vxvy = np.ascontiguousarray(pts[:, :2], np.int32), np.ascontiguousarray(pts[:, 2:], np.float32)
    nu = np.round(rng.uniform(5, 50, len(pts))).astype(np.float32)
    for ms in (1, 3):
        want_l, want_r = orc.cluster_candidates(x0y0, vxvy, nu, 2.5, 4.5, ms)
        label, rep = kb.cluster_candidates(_cuda(x0y0), _cuda(vxvy), _cuda(nu), 2.5, 4.5, ms)
        assert (label.cpu().numpy() == want_l).all() and (rep.cpu().numpy() == want_r).all()
    cfg = synth.config(1)
    st = synth.make_stack(cfg)
    pp = kb.make_psi_phi(_cuda(st.sci), _cuda(st.var), _cuda(st.mask), st.psf)
    count, got = kb.search_threshold(pp, st.times, st.vel_grid, cfg.min_obs, 12.0, 4096)
    n = int(count.item())
    assert 2 <= n <= 4096
    xy = torch.stack([got["x"][:n], got["y"][:n]], 1).contiguous()
    vel = _cuda(st.vel_grid)[got["vel_idx"][:n].long()].contiguous()
    label, rep = kb.cluster_candidates(xy, vel, got["nu"][:n].contiguous(), 3.0, 8.0, 1)
    keep = rep.cpu().numpy() == 1
    assert 1 <= keep.sum() <= n // 8          # hundreds of near-duplicates collapse to a handful of groups
    b = int(torch.argmax(got["nu"][:n]).item())
    assert keep[b] and abs(int(got["x"][b]) - 20) <= 1 and abs(int(got["y"][b]) - 30) <= 1
