"""Device-side logic of the direct-gather search (top-K and threshold forms) and of the kernels
around the search (csrc/postproc.cu: N1 light-curve filter, N2 stamps and moments, N3 mask builder;
threshold mode of the queued tiled kernel), run WITHOUT a GPU under the SIMT emulator of
tests/hostlogic/simt/ on exact-size buffers, against the CPU oracle: bit for bit, every output.
The same file runs under AddressSanitizer + UBSan in tests/test_simt_sanitized.py.
"""
import ctypes
import math

import numpy as np
import pytest

from paper_1901_02492_b200 import synth
from tests import simt_build

PLANES = ("vel_idx", "n_obs", "psi", "phi", "nu", "alpha")
CAND_I, CAND_F = ("x", "y", "vel_idx", "n_obs"), ("psi", "phi", "nu", "alpha")
ptr = lambda a: None if a is None else a.ctypes.data_as(ctypes.c_void_p)


@pytest.fixture(scope="module")
def sim():
    return simt_build.load("post_simt")


@pytest.fixture(scope="module")
def simt_tiled():
    return simt_build.load("tiled_simt")


def bits_equal(a, b):
    return ((a.view(np.int32) == b.view(np.int32)) | (a == b)).all() if a.dtype == np.float32 else (a == b).all()


# ------------------------------------------------------------------------------ S1 + S2
def run_psi_phi(sim, sci, var, mask, psf, misalign=0):
    N, H, W = sci.shape
    sci, var, psf = (np.ascontiguousarray(a, np.float32) for a in (sci, var, psf))
    out = np.zeros((N, H, W, 2), np.float32)
    launches = ctypes.c_int(0)
    rc = sim.simt_make_psi_phi(ptr(sci), ptr(var), ptr(mask), ptr(psf), N, H, W, psf.shape[-1], ptr(out), misalign,
                               ctypes.byref(launches), 2, ctypes.c_uint(7))
    assert rc == 0
    return out, launches.value


def assert_psiphi_close(gpu, ref, pabs):
    gn, rn = np.isnan(gpu[..., 0]), np.isnan(ref[..., 0])
    assert (gn == rn).all() and (gpu[..., 1][rn] == 0).all()
    ok = ~rn
    assert (np.abs(gpu[..., 0][ok] - ref[..., 0][ok]) <= 1e-5 * pabs[ok] + 1e-7).all()
    assert (np.abs(gpu[..., 1][ok] - ref[..., 1][ok]) <= 1e-5 * ref[..., 1][ok] + 1e-7).all()


@pytest.mark.parametrize("k,over", [
    (1, {}),                                           # 64 x 64, P = 11: exactly one tile per image
    (2, dict(N=3, H=70, W=132)),                       # several tiles + ragged tail, P = 19, W % 4 == 0
    (4, dict(N=2, H=40, W=68, n_sources=3)),           # elliptical PSF, P = 27, 10 % static mask
    (3, dict(N=2, H=37, W=67, n_sources=2)),           # odd width: the scalar path is the only one
])
def test_psi_phi_vector_and_scalar_paths(sim, orc, k, over):
    """psi_phi_kernel in one launch for the stack: within the section 8(c) tolerance of the oracle,
    and the float4 stage / coalesced store path bit-identical to the scalar path (round 1's)."""
    st = synth.make_stack(synth.config(k, **over))
    ref, pabs = orc.make_psi_phi(st.sci, st.var, st.mask, st.psf, want_abs=True)
    vec, n_launch = run_psi_phi(sim, st.sci, st.var, st.mask, st.psf)
    assert n_launch == 1, "the whole stack goes in one launch"
    assert_psiphi_close(vec, ref, pabs)
    scalar, _ = run_psi_phi(sim, st.sci, st.var, st.mask, st.psf, misalign=1)
    assert (vec.view(np.int32) == scalar.view(np.int32)).all()
    nomask, _ = run_psi_phi(sim, st.sci, st.var, None, st.psf)
    ref2, pabs2 = orc.make_psi_phi(st.sci, st.var, None, st.psf, want_abs=True)
    assert_psiphi_close(nomask, ref2, pabs2)


def test_psi_phi_many_images_split_into_launches_and_bad_numerics(sim, orc):
    """P = 31 takes 8 images per launch: 19 images need 3 launches; bad numerics and 1 x 1 PSFs."""
    rng = np.random.default_rng(0)
    sci = rng.standard_normal((19, 9, 12)).astype(np.float32)
    var = rng.uniform(1, 2, (19, 9, 12)).astype(np.float32)
    sci[0, 1, 1] = np.nan; sci[1, 2, 3] = np.inf; var[0, 3, 3] = 0.0; var[18, 0, 0] = -1.0; var[7, 8, 11] = np.inf
    mask = (rng.random((19, 9, 12)) < 0.1).astype(np.uint8)
    for P, want_launches in ((31, 3), (1, 1), (5, 1)):
        psf = rng.uniform(0.0, 1.0, (19, P, P)).astype(np.float32)
        ref, pabs = orc.make_psi_phi(sci, var, mask, psf, want_abs=True)
        got, n_launch = run_psi_phi(sim, sci, var, mask, psf)
        assert n_launch == want_launches
        assert_psiphi_close(got, ref, pabs)


# ------------------------------------------------------------------------------ direct search
def run_direct(sim, pp, times, vel, K, mo, y0=0, y1=None, order=0, seed=1):
    N, H, W, _ = pp.shape
    y1 = H if y1 is None else y1
    pp, times, vel = (np.ascontiguousarray(pp, np.float32), np.ascontiguousarray(times, np.float64),
                      np.ascontiguousarray(vel, np.float32))
    out = {k: np.full((y1 - y0, W, K), -77, np.int32 if k in PLANES[:2] else np.float32) for k in PLANES}
    rc = sim.simt_search_direct(ptr(pp), ptr(times), N, H, W, ptr(vel), int(vel.shape[0]), K, mo, y0, y1,
                                *[ptr(out[k]) for k in PLANES], order, ctypes.c_uint(seed))
    assert rc == 0
    return out


def test_direct_search_matches_the_oracle_exactly(sim, orc):
    """search_direct_kernel after the round-2 changes (row band, insert rule of topk_list.h): config 1
    whole, a K = 16 crop, bands, duplicated velocities, fewer eligible than K, all-invalid stack."""
    cfg = synth.config(1)
    st = synth.make_stack(cfg)
    pp = orc.make_psi_phi(st.sci, st.var, st.mask, st.psf)
    ref = orc.search(pp, st.times, st.vel_grid, cfg.K, cfg.min_obs)
    out = run_direct(sim, pp, st.times, st.vel_grid, cfg.K, cfg.min_obs, order=2, seed=3)
    for k in PLANES:
        assert bits_equal(out[k], ref[k]), k
    for y0, y1 in ((0, 8), (7, 33), (63, 64), (20, 20)):
        band = run_direct(sim, pp, st.times, st.vel_grid, cfg.K, cfg.min_obs, y0, y1)
        for k in PLANES:
            assert bits_equal(band[k], ref[k][y0:y1]), k
    pp = synth.random_psiphi(5, 37, 70, seed=3, invalid_frac=0.1)
    vel = synth.velocity_grid(4, 4, -2, 2, 2, 12)
    vel = np.concatenate([vel, vel[3:9], vel[:2]])
    times = np.array([5.0, 4.5, 6.0, 5.25, 7.0])
    for K, mo in ((8, 2), (16, 5), (32, 1), (3, 3)):
        out, ref = run_direct(sim, pp, times, vel, K, mo, order=1), orc.search(pp, times, vel, K, mo)
        for k in PLANES:
            assert bits_equal(out[k], ref[k]), (k, K)
    # a candidate whose nu is -inf (Psi = -inf) still takes an empty slot, as in the oracle
    pp = synth.random_psiphi(2, 6, 33, seed=9, invalid_frac=0.0)
    pp[0, :, ::3, 0] = -np.inf
    out, ref = run_direct(sim, pp, [0.0, 1.0], vel[:5], 4, 1), orc.search(pp, [0.0, 1.0], vel[:5], 4, 1)
    assert np.isneginf(ref["nu"][ref["vel_idx"] >= 0]).any()
    for k in PLANES:
        assert bits_equal(out[k], ref[k]), k
    pp = synth.random_psiphi(3, 9, 40, seed=2, invalid_frac=1.0)
    out = run_direct(sim, pp, [0.0, 1.0, 2.0], vel[:5], 4, 1)
    assert (out["vel_idx"] == -1).all() and np.isneginf(out["nu"]).all() and (out["n_obs"] == 0).all()


# ------------------------------------------------------------------------------ N4
def run_threshold(lib, fn, pp, times, vel, mo, nu_min, cap, y0=0, y1=None, order=2, seed=5):
    N, H, W, _ = pp.shape
    y1 = H if y1 is None else y1
    pp, times, vel = (np.ascontiguousarray(pp, np.float32), np.ascontiguousarray(times, np.float64),
                      np.ascontiguousarray(vel, np.float32))
    out = {k: np.zeros(max(cap, 1), np.int32) for k in CAND_I}
    out.update({k: np.zeros(max(cap, 1), np.float32) for k in CAND_F})
    f = getattr(lib, fn)
    f.restype = ctypes.c_longlong
    n = f(ptr(pp), ptr(times), N, H, W, ptr(vel), int(vel.shape[0]), mo, ctypes.c_float(nu_min), y0, y1,
          ctypes.c_longlong(cap), *[ptr(out[k]) for k in CAND_I + CAND_F], order, ctypes.c_uint(seed))
    assert n >= 0, f"{fn} returned {n}"
    return int(n), {k: v[:min(n, cap)] for k, v in out.items()}


def sorted_records(c):
    order = np.lexsort((c["vel_idx"], c["x"], c["y"]))
    return {k: v[order] for k, v in c.items()}


@pytest.mark.parametrize("which", ["direct", "tiled"])
def test_threshold_search_emits_exactly_the_oracle_set(sim, simt_tiled, orc, which):
    lib, fn = (sim, "simt_search_direct_threshold") if which == "direct" else (simt_tiled, "simt_search_tiled_threshold")
    cfg = synth.config(1)
    st = synth.make_stack(cfg)
    pp = orc.make_psi_phi(st.sci, st.var, st.mask, st.psf)
    cases = [(pp, st.times, st.vel_grid, cfg.min_obs, 4.0, 0, cfg.H), (pp, st.times, st.vel_grid, 1, 2.5, 9, 41)]
    pp2 = synth.random_psiphi(9, 100, 140, seed=21, invalid_frac=0.03)      # interior tiles, many candidates
    t2 = np.array([0, .05, .1, .15, 1, 1.05, 1.1, 2.0, 2.05])
    v2 = synth.velocity_grid(6, 5, -math.pi / 3, math.pi / 3, 3.0, 40.0)
    cases += [(pp2, t2, v2, 5, 1.0, 0, 100), (pp2, t2, v2, 9, -1e30, 30, 70)]
    pp3 = synth.random_psiphi(20, 40, 97, seed=6, invalid_frac=0.2)          # N > 16: additive counters
    t3 = np.sort(np.random.default_rng(3).uniform(0, 3, 20))
    cases += [(pp3, t3, synth.velocity_grid(4, 4, -1, 1, 1, 30), 6, 0.5, 0, 40)]
    for pp_, t_, v_, mo, thr, y0, y1 in cases:
        n_ref, ref = orc.search_threshold(pp_, t_, v_, mo, thr, y0, y1)
        n, got = run_threshold(lib, fn, pp_, t_, v_, mo, thr, n_ref + 7, y0, y1)
        assert n == n_ref and n > 0
        got, ref = sorted_records(got), sorted_records(ref)
        for k in CAND_I + CAND_F:
            assert bits_equal(got[k], ref[k]), k
        # capacity below the count: the count stays exact, nothing is written past the capacity
        n2, part = run_threshold(lib, fn, pp_, t_, v_, mo, thr, 3, y0, y1)
        assert n2 == n_ref and len(part["nu"]) == min(3, n_ref)
    n, _ = run_threshold(lib, fn, pp, st.times, st.vel_grid, cfg.min_obs, 1e30, 4)
    assert n == 0


# ------------------------------------------------------------------------------ N1
def run_filter(sim, pp, times, x0y0, vxvy, sigma=5.0, q=0.0, order=2):
    N, H, W, _ = pp.shape
    M = len(x0y0)
    pp, times = np.ascontiguousarray(pp, np.float32), np.ascontiguousarray(times, np.float64)
    x0y0, vxvy = np.ascontiguousarray(x0y0, np.int32), np.ascontiguousarray(vxvy, np.float32)
    out = {k: np.zeros(M, np.float32) for k in ("psi", "phi", "nu", "alpha")}
    out["n_obs"], out["keep"], out["kalman"] = np.zeros(M, np.int32), np.zeros(M, np.uint64), np.zeros((M, 2), np.float32)
    rc = sim.simt_filter_candidates(ptr(pp), ptr(times), N, H, W, ptr(x0y0), ptr(vxvy), M, ctypes.c_float(sigma),
                                    ctypes.c_float(q), *[ptr(out[k]) for k in ("psi", "phi", "n_obs", "nu", "alpha", "keep", "kalman")],
                                    order, ctypes.c_uint(1))
    assert rc == 0
    return out


def test_filter_candidates_matches_the_oracle_bit_for_bit(sim, orc):
    rng = np.random.default_rng(17)
    for N, frac, q, sigma in ((8, 0.0, 0.0, 5.0), (15, 0.1, 0.0, 5.0), (15, 0.1, 3.5, 3.0), (64, 0.3, 0.25, 2.0), (1, 0.0, 0.0, 5.0)):
        H, W, M = 50, 80, 700
        pp = synth.random_psiphi(N, H, W, seed=100 + N, invalid_frac=frac)
        pp[..., 1] = np.where(rng.random((N, H, W)) < 0.02, 0.0, pp[..., 1])      # Phi_i = 0 with valid psi
        spikes = rng.random((N, H, W)) < 0.05                                      # outliers to reject
        pp[..., 0] = np.where(spikes, pp[..., 0] * 60.0, pp[..., 0])
        times = np.sort(rng.uniform(0, 3.0, N))
        x0y0 = np.stack([rng.integers(0, W, M), rng.integers(0, H, M)], 1).astype(np.int32)
        vxvy = rng.uniform(-12, 12, (M, 2)).astype(np.float32)
        vxvy[:50] = 0.0
        ref = orc.filter_candidates(pp, times, x0y0, vxvy, sigma, q)
        got = run_filter(sim, pp, times, x0y0, vxvy, sigma, q)
        assert (got["keep"] == ref["keep"]).all() and (got["n_obs"] == ref["n_obs"]).all()
        for k in ("psi", "phi", "nu", "alpha", "kalman"):
            assert bits_equal(got[k], ref[k]), (k, N)
        if N >= 8:
            full = np.array([bin(int(k)).count("1") for k in ref["keep"]])
            assert (full < N).any() and (ref["n_obs"] > 0).any(), "the case must exercise rejections"


# ------------------------------------------------------------------------------ N2
def test_coadd_stamps_and_moments_match_the_oracle_bit_for_bit(sim, orc):
    rng = np.random.default_rng(23)
    N, H, W = 7, 45, 60
    sci = rng.normal(0, 10, (N, H, W)).astype(np.float32)
    sci[:, 20:25, 30:35] += 300.0
    sci[2, 22, 31] = np.nan
    mask = (rng.random((N, H, W)) < 0.05).astype(np.uint8)
    times = np.sort(rng.uniform(0, 2.0, N))
    M = 40
    x0y0 = np.stack([rng.integers(0, W, M), rng.integers(0, H, M)], 1).astype(np.int32)
    x0y0[:4] = [[0, 0], [W - 1, H - 1], [32, 22], [59, 0]]
    vxvy = rng.uniform(-6, 6, (M, 2)).astype(np.float32)
    vxvy[2] = 0.0
    keep = rng.integers(0, 1 << N, M).astype(np.uint64)
    keep[2] = (1 << N) - 1
    for R, msk, kp in ((10, mask, keep), (3, None, None), (0, mask, None), (15, None, keep)):
        S = 2 * R + 1
        st_ref, mo_ref = orc.coadd_stamps(sci, msk, times, x0y0, vxvy, kp, R)
        st = np.zeros((M, S, S), np.float32)
        mo = np.zeros((M, 6), np.float32)
        rc = sim.simt_coadd_stamps(ptr(sci), ptr(msk), ptr(times), N, H, W, ptr(x0y0), ptr(vxvy), ptr(kp), M, R,
                                   ptr(st), ptr(mo), 2, ctypes.c_uint(R + 1))
        assert rc == 0
        assert bits_equal(st, st_ref) and bits_equal(mo, mo_ref), R
    assert mo_ref[2, 0] > 0 and abs(mo_ref[2, 1]) < 2.0


# ------------------------------------------------------------------------------ N3
def test_build_mask_matches_the_oracle_exactly(sim, orc):
    rng = np.random.default_rng(29)
    for (N, H, W, grow, mi) in ((4, 50, 70, 2, 2), (3, 33, 31, 0, 1), (6, 70, 100, 8, 3), (1, 5, 5, 3, 1)):
        var = rng.uniform(80, 150, (N, H, W)).astype(np.float32)
        sci = (rng.normal(0, 1, (N, H, W)) * np.sqrt(var) * 2.2).astype(np.float32)      # a few % above 5 sigma... of var
        for _ in range(6):
            y, x = rng.integers(0, H), rng.integers(0, W)
            sci[:, y, x] += 500.0
        sci[0, 0, 0] = np.nan
        var[0, H - 1, W - 1] = -1.0
        mask_in = (rng.random((N, H, W)) < 0.01).astype(np.uint8)
        for m_in in (mask_in, None):
            want = orc.build_mask(sci, var, m_in, 5.0, grow, mi, 120.0)
            got = np.zeros((N, H, W), np.uint8)
            rc = sim.simt_build_mask(ptr(sci), ptr(var), ptr(m_in), N, H, W, ctypes.c_float(5.0), grow, mi,
                                     ctypes.c_float(120.0), ptr(got), 1, ctypes.c_uint(1))
            assert rc == 0 and (got == want).all()
            assert want.any() and (H < 10 or not want.all())


# ------------------------------------------------------------------------------ N5
def test_cluster_candidates_matches_the_oracle_exactly(sim, orc):
    """DBSCAN by min-label propagation + pointer jumping: same canonical labels and representatives
    as the oracle's flood fill, incl. chains (many propagation rounds), border points, noise, ties."""
    rng = np.random.default_rng(61)
    cases = []
    centres = np.stack([rng.integers(0, 300, 30), rng.integers(0, 300, 30), rng.integers(-30, 30, 30) * 4,
                        rng.integers(-30, 30, 30) * 4], 1)
    pts = np.concatenate([centres[rng.integers(0, 30, 600)] +
                          np.stack([rng.integers(-2, 3, 600), rng.integers(-2, 3, 600), rng.integers(-2, 3, 600) * 2,
                                    rng.integers(-2, 3, 600) * 2], 1),
                          np.stack([rng.integers(0, 300, 70), rng.integers(0, 300, 70), rng.integers(-120, 120, 70),
                                    rng.integers(-120, 120, 70)], 1)])
    cases.append((pts, 2.5, 4.5))
    chain = np.stack([np.arange(700)[::-1] * 2, np.zeros(700, int), np.zeros(700, int), np.zeros(700, int)], 1)   # one long chain
    cases.append((chain, 2.0, 1.0))
    cases.append((np.array([[5, 5, 0, 0]]), 1.0, 1.0))
    for pts, exy, ev in cases:
        x0y0, vxvy = np.ascontiguousarray(pts[:, :2], np.int32), np.ascontiguousarray(pts[:, 2:], np.float32)
        M = len(pts)
        nu = np.round(rng.uniform(5, 50, M)).astype(np.float32)             # rounded: exact ties occur
        for ms in (1, 3):
            want_l, want_r = orc.cluster_candidates(x0y0, vxvy, nu, exy, ev, ms)
            label, rep, n = np.zeros(M, np.int32), np.zeros(M, np.uint8), ctypes.c_int(0)
            rc = sim.simt_cluster_candidates(ptr(x0y0), ptr(vxvy), ptr(nu), M, ctypes.c_float(exy), ctypes.c_float(ev), ms,
                                             ptr(label), ptr(rep), ctypes.byref(n), 2, ctypes.c_uint(ms))
            assert rc == 0 and (label == want_l).all() and (rep == want_r).all()
        if M == 700:
            assert n.value < 60, "pointer jumping: a chain of 700 must not need 700 rounds"
