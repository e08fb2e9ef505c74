"""Pins that check the CPU oracle against things other than itself (CPU only).

P1 analytic source, P2 N(0,1) statistics, P3 v=0 coadd == numpy.average, P4 independent
brute force, P5 index-revealing images + hand-derived literals, P6 mask invariants,
P7 scalings/symmetries, plus orientation (correlation vs convolution) and top-K rules.
"""
import math
import os

import numpy as np
import pytest

from paper_1901_02492_b200 import synth
from tests import brute

GOLDEN = os.path.join(os.path.dirname(__file__), "golden")


def _golden_kv(name):
    out = {}
    for line in open(os.path.join(GOLDEN, name)):
        line = line.split("#")[0].split()
        if len(line) == 2:
            out[line[0]] = float(line[1])
    return out


def _golden_rows(name):
    rows = []
    for line in open(os.path.join(GOLDEN, name)):
        line = line.split("#")[0].split()
        if len(line) == 4:
            rows.append((int(line[0]), float(line[1]), float(line[2]), int(line[3])))
    return rows


def _gauss_psf(sigma, P):
    return synth.gaussian_psf_kernels([sigma], [sigma], [0.0], P)[0]


# ------------------------------------------------------------------------------ P1
def test_p1_analytic_source_config1(orc):
    """Noiseless F*T on integer pixels along the true track: alpha = F, nu = F sqrt(N sumT2)/sigma."""
    g = _golden_kv("p1_analytic.txt")
    N, H, W, P = 5, 64, 64, 11
    T = _gauss_psf(1.0, P)
    assert abs(float((T.astype(np.float64) ** 2).sum()) - g["sumT2"]) < 5e-7
    times = np.array([0.0, 0.1, 0.2, 1.0, 1.1])
    # a velocity whose positions are integers at every epoch: fl(10*dt) in {0,1,2,10,11}
    v = np.array([[10.0, -10.0]], np.float32)
    sci = np.zeros((N, H, W), np.float32)
    x0, y0 = 20, 30
    r = P // 2
    track = []
    for i in range(N):
        dx = int(round(10.0 * times[i]))
        dy = -dx
        track.append((x0 + dx, y0 + dy))
        sci[i, y0 + dy - r:y0 + dy + r + 1, x0 + dx - r:x0 + dx + r + 1] += 500.0 * T
    var = np.full((N, H, W), 100.0, np.float32)
    psf = np.stack([T] * N)
    pp = orc.make_psi_phi(sci, var, None, psf)
    Psi, Phi, nobs, ixiy = orc.eval_trajectories(pp, times, [[x0, y0]], v, mode=orc.MODE_F64)
    assert [tuple(p) for p in ixiy[0]] == track
    nu, alpha = orc.score(Psi, Phi)
    assert nobs[0] == N
    assert abs(alpha[0] - g["alpha"]) < 5e-3
    assert abs(nu[0] - g["nu"]) < 5e-4
    # and through the search: best candidate of the start pixel when v is on the grid
    # (grid node 3 = (9.60,-9.60) px/day rounds to the same pixels: an exact tie, smaller index first)
    grid = synth.velocity_grid(8, 8, -math.pi / 4, math.pi / 4, 5, 25)
    res = orc.search(pp, times, np.concatenate([grid, v]), 4, 3)
    assert list(res["vel_idx"][y0, x0, :2]) == [3, 64]
    assert res["nu"][y0, x0, 0] == res["nu"][y0, x0, 1]
    assert abs(res["nu"][y0, x0, 0] - g["nu"]) < 5e-4
    assert res["nu"][y0, x0, 0] == res["nu"].max()


def test_p1_subpixel_direct_sum(orc):
    """Sub-pixel injection (the generator's config-1 source): Psi_i = (F/s2) sum_x T(x-s_i) T(x-y_i)
    evaluated independently in float64."""
    cfg = synth.config(1)
    st = synth.make_stack(cfg, noise=False)
    pp = orc.make_psi_phi(st.sci, st.var, st.mask, st.psf)
    v = np.array([[12.0, -4.0]], np.float32)
    Psi, Phi, nobs, ixiy = orc.eval_trajectories(pp, st.times, [[20, 30]], v, mode=orc.MODE_F64)
    F, s2, sig = 500.0, 100.0, 1.0
    T = st.psf[0].astype(np.float64)
    r = T.shape[0] // 2
    ePsi = ePhi = 0.0
    for i in range(cfg.N):
        dt = st.times[i]
        sx, sy = 20.0 + 12.0 * dt, 30.0 - 4.0 * dt
        ix, iy = ixiy[0, i]
        assert abs(ix - sx) <= 0.5 + 1e-9 and abs(iy - sy) <= 0.5 + 1e-9
        # generator's source model: unit-sum Gaussian sampled at pixel centres around (sx, sy)
        rad = 6
        cx, cy = int(math.floor(sx + 0.5)), int(math.floor(sy + 0.5))
        xs = np.arange(cx - rad, cx + rad + 1)
        ys = np.arange(cy - rad, cy + rad + 1)
        g = np.exp(-0.5 * (((xs[None, :] - sx) / sig) ** 2 + ((ys[:, None] - sy) / sig) ** 2))
        g *= F / g.sum()
        for a, yy in enumerate(ys):
            for b, xx in enumerate(xs):
                ddx, ddy = xx - ix, yy - iy
                if abs(ddx) <= r and abs(ddy) <= r:
                    ePsi += float(np.float32(g[a, b])) / s2 * T[ddy + r, ddx + r]
        ePhi += (T ** 2).sum() / s2
    assert abs(Psi[0] - ePsi) <= 2e-6 * abs(ePsi)
    assert abs(Phi[0] - ePhi) <= 2e-6 * abs(ePhi)
    nu, alpha = orc.score(Psi, Phi)
    assert 30.0 < nu[0] < 31.5 and 470.0 < alpha[0] < 500.0     # ~30.62, ~485.3


# ------------------------------------------------------------------------------ P2
def test_p2_noise_gives_unit_normal_nu(orc):
    """sci ~ N(0,var) with masks and edges: every trajectory's nu ~ N(0,1)."""
    from scipy import stats
    cfg = synth.config(2, N=6, H=96, W=128, n_sources=0, mask_frac=0.05,
                       n_angles=4, n_speeds=3, speed_lo=20.0, speed_hi=60.0)
    st = synth.make_stack(cfg, seed=11)
    pp = orc.make_psi_phi(st.sci, st.var, st.mask, st.psf)
    Psi, Phi, nobs = orc.eval_all(pp, st.times, st.vel_grid, mode=orc.MODE_F64)
    ok = (nobs >= 1) & (Phi > 0)
    nu, _ = orc.score(Psi[ok], Phi[ok])
    assert nu.size > 1e5
    assert abs(nu.mean()) < 0.02
    assert abs(nu.std() - 1.0) < 0.02
    # thinned (one start pixel per 9x9 block, one velocity): nearly independent samples
    thin = nu_thin = None
    Psi1, Phi1, n1 = Psi[4::9, 4::9, 5], Phi[4::9, 4::9, 5], nobs[4::9, 4::9, 5]
    sel = (n1 >= 1) & (Phi1 > 0)
    nu_thin, _ = orc.score(Psi1[sel], Phi1[sel])
    assert stats.kstest(nu_thin, "norm").pvalue > 1e-3
    # per-image single-pixel statistic too: Var(Psi) = Phi pixel by pixel
    z = pp[..., 0] / np.sqrt(np.where(pp[..., 1] > 0, pp[..., 1], 1))
    z = z[np.isfinite(z)]
    assert abs(z.std() - 1.0) < 0.01 and abs(z.mean()) < 0.01


# ------------------------------------------------------------------------------ P3
def test_p3_zero_velocity_is_inverse_variance_coadd(orc):
    """v = 0 with the 1x1 PSF [1]: alpha = numpy.average(sci, weights=1/var), nu = alpha sqrt(sum 1/var)."""
    rng = np.random.default_rng(5)
    N, H, W = 7, 24, 40
    var = rng.uniform(50, 400, size=(N, H, W)).astype(np.float32)
    sci = (rng.standard_normal((N, H, W)) * np.sqrt(var) + 3.0).astype(np.float32)
    psf = np.ones((N, 1, 1), np.float32)
    times = np.sort(rng.uniform(0, 3, N))
    pp = orc.make_psi_phi(sci, var, None, psf)
    res = orc.search(pp, times, np.zeros((1, 2), np.float32), 1, 1, mode=orc.MODE_F64)
    w = 1.0 / var.astype(np.float64)
    alpha = np.average(sci.astype(np.float64), weights=w, axis=0)
    nu = alpha * np.sqrt(w.sum(axis=0))
    assert (res["n_obs"][..., 0] == N).all() and (res["vel_idx"][..., 0] == 0).all()
    np.testing.assert_allclose(res["alpha"][..., 0], alpha, rtol=2e-6, atol=1e-6)
    np.testing.assert_allclose(res["nu"][..., 0], nu, rtol=2e-6, atol=1e-6)


# ------------------------------------------------------------------------------ P4
@pytest.mark.parametrize("seed", [0, 1, 2])
def test_p4_brute_force_tiny(orc, seed):
    rng = np.random.default_rng(100 + seed)
    N, H, W, K = 4, 9, 11, 3
    pp = synth.random_psiphi(N, H, W, seed=200 + seed, invalid_frac=0.15)
    times = np.array([0.0, 0.25, 0.5, 1.25]) + 0.125 * seed
    # velocities whose v*dt stay far (>= 1/16 px) from pixel boundaries: multiples of 1/4 px/day
    # times multiples of 1/4 day give multiples of 1/16 px; avoid exact k+1/2 by an odd 1/32 shift
    vel = (rng.integers(-24, 25, size=(7, 2)) / 4.0 + 1.0 / 32.0).astype(np.float32)
    vel[3] = vel[1]                                    # duplicate entry -> tie-break by index
    ref = brute.search(pp, times, vel, K, min_obs=2)
    for mode in (orc.MODE_F64, orc.MODE_F32SEQ):
        res = orc.search(pp, times, vel, K, 2, mode=mode)
        assert (res["vel_idx"] == ref["vel_idx"]).all()
        assert (res["n_obs"] == ref["n_obs"]).all()
        real = ref["vel_idx"] >= 0
        for k in ("psi", "phi", "nu", "alpha"):
            np.testing.assert_allclose(res[k][real], ref[k][real], rtol=3e-6, atol=1e-6)
        assert np.isneginf(res["nu"][~real]).all()
        for k in ("psi", "phi", "alpha", "n_obs"):
            assert (res[k][~real] == 0).all()
        if mode == orc.MODE_F32SEQ:
            # the bit-level definition of f32seq (Q18; Eq.24-25): binary32 adds in
            # image order, then correctly rounded sqrt and divisions -- a reversed or pairwise order,
            # or a double accumulator rounded once, fails this on the random stacks
            for k in ("psi", "phi", "nu", "alpha"):
                assert (res[k].view(np.int32) == ref[k + "32"].view(np.int32)).all(), k
    assert (~(ref["vel_idx"] >= 0)).any() and (ref["vel_idx"] >= 0).any()


# ------------------------------------------------------------------------------ P5
def test_p5_golden_index_literals(orc):
    rows = _golden_rows("p5_index_cases.txt")
    assert len(rows) >= 14
    n = 4096
    pp = np.zeros((2, 1, n, 2), np.float32)
    pp[1, 0, :, 0] = np.arange(n, dtype=np.float32)
    pp[..., 1] = 1.0
    for p0, v, dt, want in rows:
        times = np.array([0.0, dt])
        # x axis
        Psi, Phi, nobs, ixiy = orc.eval_trajectories(pp, times, [[p0, 0]], [[v, 0.0]])
        if 0 <= want < n:
            assert ixiy[0, 1, 0] == want and Psi[0] == want and nobs[0] == 2, (p0, v, dt)
        else:
            assert ixiy[0, 1, 0] == -1 and nobs[0] == 1, (p0, v, dt)
        # y axis (same rule): transpose the image
        ppT = np.ascontiguousarray(pp.transpose(0, 2, 1, 3))
        Psi, Phi, nobs, ixiy = orc.eval_trajectories(ppT, times, [[0, p0]], [[0.0, v]])
        if 0 <= want < n:
            assert ixiy[0, 1, 1] == want and Psi[0] == want, (p0, v, dt)
        else:
            assert ixiy[0, 1, 1] == -1 and nobs[0] == 1, (p0, v, dt)


def test_p5_index_revealing_images(orc):
    """psi_1[y,x] = y*W+x, phi = 1, image 0 zero: Psi IS the sampled linear index."""
    H, W = 37, 53
    pp = np.zeros((2, H, W, 2), np.float32)
    pp[1, ..., 0] = (np.arange(H)[:, None] * W + np.arange(W)[None, :]).astype(np.float32)
    pp[..., 1] = 1.0
    times = np.array([10.0, 10.5])
    vel = np.array([[7.0, -3.0], [-5.0, 9.0], [2.0, 2.0], [-1.0, -1.0], [0.0, 0.0]], np.float32)
    Psi, Phi, nobs = orc.eval_all(pp, times, vel)
    for j, (vx, vy) in enumerate(vel):
        ox = math.floor(vx * 0.5 + 0.5)      # exact in binary arithmetic: halves round up
        oy = math.floor(vy * 0.5 + 0.5)
        for y0 in range(H):
            for x0 in range(W):
                ix, iy = x0 + ox, y0 + oy
                if 0 <= ix < W and 0 <= iy < H:
                    assert Psi[y0, x0, j] == iy * W + ix and nobs[y0, x0, j] == 2
                else:
                    assert Psi[y0, x0, j] == 0 and nobs[y0, x0, j] == 1


# ------------------------------------------------------------------------------ orientation
def test_correlation_orientation_asymmetric_psf(orc):
    """Eq.19 is a cross-correlation: Psi(y) = sum_d s(y+d) T(d).  One off-centre tap pins it."""
    N, H, W, P = 1, 16, 16, 5
    psf = np.zeros((N, P, P), np.float32)
    psf[0, 2 + 1, 2 + 2] = 1.0                  # T(dx=+2, dy=+1) = 1
    psf[0, 2, 2] = 0.5                          # centre tap so Phi(centre) > 0
    sci = np.zeros((N, H, W), np.float32)
    sci[0, 8, 9] = 40.0
    var = np.full((N, H, W), 4.0, np.float32)
    pp = orc.make_psi_phi(sci, var, None, psf)
    # Psi(y) picks s(y + d): the tap contributes at y = x_src - d = (9-2, 8-1)
    assert pp[0, 7, 7, 0] == pytest.approx(10.0)
    assert pp[0, 8, 9, 0] == pytest.approx(5.0)
    assert pp[0, 9, 11, 0] == 0.0
    assert pp[0, 5, 5, 1] == pytest.approx((1.0 + 0.25) / 4.0)
    # borders: out-of-image terms have zero weight (Phi shrinks)
    assert pp[0, 15, 15, 1] == pytest.approx(0.25 / 4.0)


# ------------------------------------------------------------------------------ P6
def test_p6_mask_invariants(orc):
    cfg = synth.config(2, N=5, H=48, W=64, n_sources=2, mask_frac=0.0,
                       n_angles=3, n_speeds=3, speed_lo=10.0, speed_hi=30.0)
    st = synth.make_stack(cfg, seed=7)
    pp0 = orc.make_psi_phi(st.sci, st.var, None, st.psf)
    r = st.psf.shape[-1] // 2
    # (a) masking one pixel changes psi/phi only inside its stencil, and invalidates the centre
    mask = np.zeros_like(st.mask)
    mask[2, 20, 30] = 1
    pp1 = orc.make_psi_phi(st.sci, st.var, mask, st.psf)
    diff = np.argwhere(~((pp0 == pp1) | (np.isnan(pp0) & np.isnan(pp1))).all(axis=-1))
    assert len(diff) > 0
    assert (diff[:, 0] == 2).all()
    assert (abs(diff[:, 1] - 20) <= r).all() and (abs(diff[:, 2] - 30) <= r).all()
    assert np.isnan(pp1[2, 20, 30, 0]) and pp1[2, 20, 30, 1] == 0.0
    assert pp1[2, 20, 31, 1] < pp0[2, 20, 31, 1]             # neighbour lost one term of Phi
    # non-finite / non-positive inputs behave like masked pixels
    sci2, var2 = st.sci.copy(), st.var.copy()
    sci2[2, 20, 30] = np.inf
    pp2 = orc.make_psi_phi(sci2, st.var, None, st.psf)
    var2[2, 20, 30] = 0.0
    pp3 = orc.make_psi_phi(st.sci, var2, None, st.psf)
    for q in (pp2, pp3):
        assert ((q == pp1) | (np.isnan(q) & np.isnan(pp1))).all()
    # (b) a fully masked image lowers every n_obs by its in-bounds hits and leaves the others' sums
    mask = np.zeros_like(st.mask)
    mask[3] = 1
    ppm = orc.make_psi_phi(st.sci, st.var, mask, st.psf)
    assert np.isnan(ppm[3, ..., 0]).all()
    A = orc.eval_all(pp0, st.times, st.vel_grid, mode=orc.MODE_F64)
    B = orc.eval_all(ppm, st.times, st.vel_grid, mode=orc.MODE_F64)
    keep = [0, 1, 2, 4]
    C = orc.eval_all(pp0[keep], st.times[keep], st.vel_grid, mode=orc.MODE_F64)
    assert (B[2] == C[2]).all() and (B[0] == C[0]).all() and (B[1] == C[1]).all()
    assert ((A[2] - B[2]) >= 0).all() and ((A[2] - B[2]) <= 1).all()
    # (c) v = 0 on an unmasked stack: n_obs = N everywhere
    Z = orc.eval_all(pp0, st.times, np.zeros((1, 2), np.float32))
    assert (Z[2] == cfg.N).all()


# ------------------------------------------------------------------------------ P7
def test_p7_scalings_and_translation(orc):
    cfg = synth.config(2, N=4, H=40, W=56, n_sources=3, mask_frac=0.02,
                       n_angles=3, n_speeds=2, speed_lo=8.0, speed_hi=20.0)
    st = synth.make_stack(cfg, seed=9)
    pp = orc.make_psi_phi(st.sci, st.var, st.mask, st.psf)
    # sci -> 4*sci (exact in binary): psi x4, phi same
    q = orc.make_psi_phi(4.0 * st.sci, st.var, st.mask, st.psf)
    ok = ~np.isnan(pp[..., 0])
    assert (q[..., 0][ok] == 4.0 * pp[..., 0][ok]).all() and (q[..., 1] == pp[..., 1]).all()
    # var -> 4*var: psi/4, phi/4, so alpha same and nu/2
    q = orc.make_psi_phi(st.sci, 4.0 * st.var, st.mask, st.psf)
    assert (q[..., 0][ok] == pp[..., 0][ok] / 4.0).all() and (q[..., 1] == pp[..., 1] / 4.0).all()
    r0 = orc.search(pp, st.times, st.vel_grid, 3, 2)
    r1 = orc.search(q, st.times, st.vel_grid, 3, 2)
    real = r0["vel_idx"] >= 0
    assert (r0["vel_idx"] == r1["vel_idx"]).all()
    assert (r1["alpha"][real] == r0["alpha"][real]).all()
    np.testing.assert_allclose(r1["nu"][real], r0["nu"][real] / 2.0, rtol=3e-7)
    # duplicated grid entry duplicates its results, adjacent, smaller index first
    vel2 = np.concatenate([st.vel_grid, st.vel_grid[2:3]])
    r2 = orc.search(pp, st.times, vel2, 7, 2)
    j = r2["vel_idx"]
    V = st.vel_grid.shape[0]
    pos2 = np.argwhere(j == 2)
    assert len(pos2) > 0
    for (y, x, k) in pos2:
        kk = np.flatnonzero(j[y, x] == V)
        assert len(kk) == 1 and kk[0] > k
        assert r2["nu"][y, x, k] == r2["nu"][y, x, kk[0]]
        # anything between them is an exact tie too, in index order
        between = j[y, x, k:kk[0] + 1]
        assert (r2["nu"][y, x, k:kk[0] + 1] == r2["nu"][y, x, k]).all()
        assert (np.diff(between) > 0).all()
    # integer translation of all images translates the psi/phi interior
    sh = 5
    sci_s = np.roll(st.sci, sh, axis=2)
    var_s = np.roll(st.var, sh, axis=2)
    m_s = np.roll(st.mask, sh, axis=2)
    qs = orc.make_psi_phi(sci_s, var_s, m_s, st.psf)
    rr = st.psf.shape[-1] // 2
    a = pp[:, :, rr:cfg.W - sh - rr]
    b = qs[:, :, rr + sh:cfg.W - rr]
    assert ((a == b) | (np.isnan(a) & np.isnan(b))).all()


def test_topk_sorted_sentinels_and_min_obs(orc):
    pp = synth.random_psiphi(5, 20, 24, seed=3, invalid_frac=0.3)
    times = np.array([0.0, 0.5, 1.0, 1.5, 2.0])
    vel = synth.velocity_grid(4, 3, -1.0, 1.0, 2.0, 9.0)
    K = 16
    r = orc.search(pp, times, vel, K, 4)
    nu = r["nu"]
    assert (nu[..., 1:] <= nu[..., :-1]).all()                   # sorted descending
    real = r["vel_idx"] >= 0
    assert (real[..., :-1] >= real[..., 1:]).all()               # sentinels only at the tail
    assert (r["n_obs"][real] >= 4).all() and (r["phi"][real] > 0).all()
    assert np.isneginf(nu[~real]).all() and (~real).any()
    # each pixel: set of kept velocities == all eligible ones when fewer than K are eligible
    Psi, Phi, nobs = orc.eval_all(pp, times, vel)
    elig = (nobs >= 4) & (Phi > 0)
    assert (real.sum(-1) == np.minimum(elig.sum(-1), K)).all()
    # f64 and f32seq agree to rounding
    r64 = orc.search(pp, times, vel, K, 4, mode=orc.MODE_F64)
    np.testing.assert_allclose(r64["nu"][real], nu[real], rtol=1e-5, atol=1e-4)


def test_times_need_not_be_sorted_and_origin_is_image0(orc):
    pp = synth.random_psiphi(3, 12, 12, seed=8, invalid_frac=0.0)
    vel = np.array([[4.0, 0.0]], np.float32)
    P1 = orc.eval_trajectories(pp, np.array([5.0, 6.0, 5.5]), [[2, 3]], vel)
    assert [tuple(p) for p in P1[3][0]] == [(2, 3), (6, 3), (4, 3)]
    P2 = orc.eval_trajectories(pp, np.array([5.0, 4.5, 6.0]), [[2, 3]], vel)
    assert [tuple(p) for p in P2[3][0]] == [(2, 3), (0, 3), (6, 3)]
