"""Pins of the oracle functions for the rows beyond the top-K search:
N4 threshold-mode search, N1 light-curve outlier filter, N3 mask builder, N2 coadded stamps and
central moments.  Each is checked against something other than itself: an independent brute force,
a closed form, a library routine (numpy.average, scipy.ndimage.binary_dilation), hand-derived
literals under tests/golden/, or an already pinned oracle function on a modified input.
Where the paper gives no parameter (filter gains, thresholds) the READING is DESIGN.md's and is
marked "parity unpinned" there; what is pinned here is that the oracle computes that reading.
"""
import math
import os

import numpy as np
import pytest
from scipy import ndimage, stats

from paper_1901_02492_b200 import synth
from tests import brute

GOLDEN = os.path.join(os.path.dirname(os.path.abspath(__file__)), "golden")


# ------------------------------------------------------------------------------------------ N4
@pytest.mark.parametrize("seed", [0, 1])
def test_n4_threshold_brute_force(orc, seed):
    """Independent Python loops (tests/brute.py, exact rational positions, full sort with K = V):
    every eligible trajectory with nu >= nu_min, nothing else, bit-identical sums."""
    rng = np.random.default_rng(300 + seed)
    N, H, W = 4, 8, 10
    pp = synth.random_psiphi(N, H, W, seed=400 + seed, invalid_frac=0.15)
    times = np.array([0.0, 0.25, 0.5, 1.25])
    vel = (rng.integers(-24, 25, size=(6, 2)) / 4.0 + 1.0 / 32.0).astype(np.float32)
    ref = brute.search(pp, times, vel, K=6, min_obs=2)
    for nu_min in (-1.0, 0.5, 1.5):
        want = sorted((int(y), int(x), int(ref["vel_idx"][y, x, k]))
                      for y in range(H) for x in range(W) for k in range(6)
                      if ref["vel_idx"][y, x, k] >= 0 and ref["nu32"][y, x, k] >= np.float32(nu_min))
        n, got = orc.search_threshold(pp, times, vel, 2, nu_min)
        assert n == len(want) and sorted(zip(got["y"], got["x"], got["vel_idx"])) == want
        for y, x, j, nu, psi, phi, al, no in zip(got["y"], got["x"], got["vel_idx"], got["nu"], got["psi"],
                                                 got["phi"], got["alpha"], got["n_obs"]):
            k = int(np.flatnonzero(ref["vel_idx"][y, x] == j)[0])
            assert nu == ref["nu32"][y, x, k] and psi == ref["psi32"][y, x, k] and phi == ref["phi32"][y, x, k]
            assert al == ref["alpha32"][y, x, k] and no == ref["n_obs"][y, x, k]
    # capacity smaller than the count: the count is still exact, the first `capacity` are stored
    n_all, _ = orc.search_threshold(pp, times, vel, 2, -1.0)
    n_cap, part = orc.search_threshold(pp, times, vel, 2, -1.0, capacity=5)
    assert n_cap == n_all > 5 and len(part["nu"]) == 5


def test_n4_noise_exceedance_rate(orc):
    """Pure N(0, var) noise: nu ~ N(0,1) per trajectory, so the number of
    trajectories above t among M is Binomial(M, Q(t)) up to their weak correlation."""
    cfg = synth.config(1, H=96, W=96, sources_explicit=(), n_angles=4, n_speeds=4)
    st = synth.make_stack(cfg)
    pp = orc.make_psi_phi(st.sci, st.var, st.mask, st.psf)
    M = 96 * 96 * 16
    for t in (2.0, 3.0):
        n, got = orc.search_threshold(pp, st.times, st.vel_grid, cfg.N, t)       # fully observed only
        _, all_ = orc.search_threshold(pp, st.times, st.vel_grid, cfg.N, -1e30)
        m_full = len(all_["nu"])
        q = stats.norm.sf(t)
        assert 0.3 * M < m_full <= M
        assert abs(n - m_full * q) < 6 * math.sqrt(m_full * q) * 3            # correlated samples: generous
        assert (got["nu"] >= t).all() and (got["n_obs"] == cfg.N).all()


# ------------------------------------------------------------------------------------------ N1
def _lightcurve_stack(f, phi=1.0):
    """A 1 x 1 pixel stack whose only trajectory (v = 0) has the light curve f with Phi_i = phi."""
    N = len(f)
    pp = np.zeros((N, 1, 1, 2), np.float32)
    pp[:, 0, 0, 1] = phi
    pp[:, 0, 0, 0] = np.asarray(f, np.float32) * np.float32(phi)
    return pp


def test_n1_golden_keep_masks(orc):
    rows = []
    for line in open(os.path.join(GOLDEN, "n1_lightcurve_cases.txt")):
        line = line.split("#")[0].strip()
        if line:
            s, q, f, bits = line.split()
            rows.append((float(s), float(q), [float(v) for v in f.split(",")], bits))
    assert len(rows) >= 12
    for s, q, f, bits in rows:
        pp = _lightcurve_stack(f)
        out = orc.filter_candidates(pp, np.arange(len(f), dtype=np.float64), [[0, 0]], [[0.0, 0.0]], s, q)
        want = int(bits, 2)                                  # written as a binary number: image 0 is the LAST digit
        assert int(out["keep"][0]) == want, (s, q, f, bits, bin(int(out["keep"][0])))
        assert out["n_obs"][0] == bits.count("1")
        kept = [v for v, b in zip(f, bits[::-1]) if b == "1"]
        assert out["psi"][0] == np.float32(sum(kept)) and out["phi"][0] == len(kept)


def test_n1_kalman_without_process_noise_is_the_weighted_mean(orc):
    """q = 0 and nothing rejected: the filter's final state is the inverse-variance weighted mean
    and its variance 1/sum(1/r) -- numpy.average is the library routine (textbook identity)."""
    rng = np.random.default_rng(5)
    N = 9
    phi = rng.uniform(0.5, 3.0, N)
    f = 10.0 + rng.normal(0, 1, N) / np.sqrt(phi)
    pp = np.zeros((N, 1, 1, 2), np.float32)
    pp[:, 0, 0, 1] = phi
    pp[:, 0, 0, 0] = f * phi
    out = orc.filter_candidates(pp, np.arange(N, dtype=np.float64), [[0, 0]], [[0.0, 0.0]], 5.0, 0.0)
    assert int(out["keep"][0]) == (1 << N) - 1
    f32 = pp[:, 0, 0, 0].astype(np.float64) / pp[:, 0, 0, 1]
    w = pp[:, 0, 0, 1].astype(np.float64)
    np.testing.assert_allclose(out["kalman"][0, 0], np.average(f32, weights=w), rtol=2e-6)
    np.testing.assert_allclose(out["kalman"][0, 1], 1.0 / w.sum(), rtol=2e-6)


@pytest.mark.parametrize("bad", [0, 4, 7])
def test_n1_rejects_exactly_the_outlier_and_rescoring_equals_s4_s5_without_it(orc, bad):
    """A moving source with one image polluted by a bright interloper (Fig.3), first, middle
    and last image: exactly that observation is dropped, and the re-scored Psi, Phi, n_obs, nu,
    alpha equal the (pinned) S4/S5 of the same trajectory on a stack where that pixel is invalid."""
    rng = np.random.default_rng(40 + bad)
    N, H, W = 8, 40, 60
    pp = synth.random_psiphi(N, H, W, seed=77, invalid_frac=0.0)
    pp[..., 1] = rng.uniform(0.04, 0.06, (N, H, W)).astype(np.float32)
    pp[..., 0] = (rng.normal(0, 1, (N, H, W)) * np.sqrt(pp[..., 1])).astype(np.float32)
    times = np.sort(rng.uniform(0, 2.0, N))
    times[0] = 0.0
    x0y0 = np.array([[10, 20], [30, 5]], np.int32)
    vxvy = np.array([[7.25, 3.5], [-4.0, 9.75]], np.float32)
    _, _, _, ixiy = orc.eval_trajectories(pp, times, x0y0, vxvy)
    flux = 50.0
    for m in range(2):
        for i in range(N):
            x, y = ixiy[m, i]
            pp[i, y, x, 0] = np.float32(flux * pp[i, y, x, 1])                # light curve = flux exactly
    clean = orc.filter_candidates(pp, times, x0y0, vxvy)
    Psi, Phi, nobs, _ = orc.eval_trajectories(pp, times, x0y0, vxvy)
    assert (clean["keep"] == (1 << N) - 1).all() and (clean["n_obs"] == N).all()
    assert (clean["psi"] == Psi).all() and (clean["phi"] == Phi).all()         # no outlier: S4 unchanged
    nu, alpha = orc.score(Psi, Phi)
    assert (clean["nu"] == nu).all() and (clean["alpha"] == alpha).all()
    x, y = ixiy[0, bad]
    pp[bad, y, x, 0] *= 40.0                                                   # flux 2000: ~ 390 sigma
    out = orc.filter_candidates(pp, times, x0y0, vxvy)
    assert int(out["keep"][0]) == ((1 << N) - 1) & ~(1 << bad) and int(out["keep"][1]) == (1 << N) - 1
    masked = pp.copy()
    masked[bad, y, x] = (np.nan, 0.0)
    Psi, Phi, nobs, _ = orc.eval_trajectories(masked, times, x0y0, vxvy)
    nu, alpha = orc.score(Psi, Phi)
    for k, ref in (("psi", Psi), ("phi", Phi), ("n_obs", nobs), ("nu", nu), ("alpha", alpha)):
        assert (out[k] == ref).all(), k


def test_n1_missing_observations_and_degenerate_light_curves(orc):
    pp = _lightcurve_stack([5, 5, 5, 5, 5, 5])
    pp[2, 0, 0] = (np.nan, 0.0)                      # invalid sample: not part of the light curve
    pp[4, 0, 0, 1] = 0.0                             # Phi_i = 0 with valid psi: untestable, stays in the sums
    out = orc.filter_candidates(pp, np.arange(6.0), [[0, 0], [0, 0]], [[0.0, 0.0], [5.0, 0.0]])
    assert int(out["keep"][0]) == 0b111011 and out["n_obs"][0] == 5 and out["phi"][0] == 4
    # second candidate leaves the 1-pixel image after image 0: one observation, never rejected
    assert int(out["keep"][1]) == 0b000001 and out["n_obs"][1] == 1 and out["nu"][1] == np.float32(5.0)
    # nothing observed at all
    pp[:] = (np.nan, 0.0)
    out = orc.filter_candidates(pp, np.arange(6.0), [[0, 0]], [[0.0, 0.0]])
    assert out["n_obs"][0] == 0 and np.isneginf(out["nu"][0]) and out["alpha"][0] == 0 and out["keep"][0] == 0


# ------------------------------------------------------------------------------------------ N3
def test_n3_mask_builder_against_scipy_morphology(orc):
    """Detection threshold, growth by a disc of radius 2 (scipy.ndimage.binary_dilation is the
    library routine), the two-image rule, the union, the bright-pixel mask."""
    rng = np.random.default_rng(8)
    N, H, W = 4, 50, 70
    var = rng.uniform(80, 150, (N, H, W)).astype(np.float32)
    sci = (rng.normal(0, 1, (N, H, W)) * np.sqrt(var)).astype(np.float32)
    static = [(10, 12), (30, 40), (0, 0), (49, 69), (25, 3)]
    for (y, x) in static:                                       # static sources: in every image
        sci[:, y, x] += 400.0
    sci[2, 20, 20] += 400.0                                     # a moving source: one image only
    sci[1, 40, 10] = 130.0                                      # above 120 counts but below 5 sigma? no: 130 > 5*sqrt(150)
    sci[3, 45, 50] = np.nan
    var[0, 5, 5] = 0.0
    mask_in = (rng.random((N, H, W)) < 0.01).astype(np.uint8)
    got = orc.build_mask(sci, var, mask_in, 5.0, 2, 2, 120.0)
    ok = np.isfinite(sci) & np.isfinite(var) & (var > 0)
    det = ok & (sci > (np.float32(5.0) * np.sqrt(var, dtype=np.float32)))
    yy, xx = np.mgrid[-2:3, -2:3]
    disc = (yy * yy + xx * xx) <= 4
    grown = np.stack([ndimage.binary_dilation(det[i], structure=disc) for i in range(N)])
    static_mask = grown.sum(0) >= 2
    want = (mask_in != 0) | static_mask[None] | (np.isfinite(sci) & (sci > 120.0))
    assert (got == want.astype(np.uint8)).all()
    assert got[:, 10, 12].all() and got[:, 12, 12].all() and not got[:, 13, 12].any()   # radius 2, not 3
    assert not got[0, 20, 20] and got[2, 20, 20]                 # moving source: only its own bright pixel
    assert got[:, 0, 0].all() and got[:, 49, 69].all()
    # min_images = 1 masks the moving source's footprint in every image; grow = 0 masks single pixels
    assert orc.build_mask(sci, var, None, 5.0, 2, 1, 1e9)[:, 21, 21].all()
    g0 = orc.build_mask(sci, var, None, 5.0, 0, 2, 1e9)
    assert g0[:, 10, 12].all() and not g0[:, 10, 13].any()


# ------------------------------------------------------------------------------------------ N2
def test_n2_stamps_are_means_over_contributing_images(orc):
    rng = np.random.default_rng(11)
    N, H, W, R = 5, 30, 40, 3
    sci = rng.normal(0, 10, (N, H, W)).astype(np.float32)
    mask = (rng.random((N, H, W)) < 0.05).astype(np.uint8)
    sci[1, 15, 20] = np.inf
    times = np.array([0.0, 0.5, 1.0, 1.5, 2.0])
    x0y0 = np.array([[20, 15], [1, 1], [38, 28]], np.int32)
    vxvy = np.array([[0.0, 0.0], [0.0, 0.0], [2.0, 1.0]], np.float32)
    keep = np.array([0b11111, 0b10101, 0b11111], np.uint64)
    stamps, _ = orc.coadd_stamps(sci, mask, times, x0y0, vxvy, keep, R)
    for m in range(3):
        for dy in range(-R, R + 1):
            for dx in range(-R, R + 1):
                vals = []
                for i in range(N):
                    if not (int(keep[m]) >> i) & 1:
                        continue
                    x = int(x0y0[m, 0] + math.floor(float(np.float32(vxvy[m, 0] * np.float32(times[i]))) + 0.5)) + dx
                    y = int(x0y0[m, 1] + math.floor(float(np.float32(vxvy[m, 1] * np.float32(times[i]))) + 0.5)) + dy
                    cx, cy = x - dx, y - dy
                    if not (0 <= cx < W and 0 <= cy < H):
                        continue                                  # the trajectory left the image
                    if 0 <= x < W and 0 <= y < H and not mask[i, y, x] and np.isfinite(sci[i, y, x]):
                        vals.append(float(sci[i, y, x]))
                want = np.mean(vals) if vals else 0.0
                assert abs(stamps[m, dy + R, dx + R] - want) <= 1e-5 * max(1.0, abs(want)), (m, dy, dx)
    # keep = None means every observation
    s2, _ = orc.coadd_stamps(sci, mask, times, x0y0[:1], vxvy[:1], None, R)
    assert (s2[0] == stamps[0]).all()


def test_n2_central_moments_against_float64_numpy(orc):
    """Moments of a sampled Gaussian: centroid and second moments equal the float64 NumPy
    weighted averages (numpy.average is the library routine); a centred circular Gaussian of
    sigma 1.5 gives cx = cy = 0, mu20 = mu02 ~ sigma^2, mu11 = 0."""
    R, S = 10, 21
    d = np.arange(-R, R + 1, dtype=np.float64)
    X, Y = np.meshgrid(d, d)
    for (cx, cy, sx, sy, rho) in ((0, 0, 1.5, 1.5, 0.0), (1.3, -0.7, 2.0, 1.2, 0.4)):
        z = ((X - cx) / sx) ** 2 - 2 * rho * (X - cx) * (Y - cy) / (sx * sy) + ((Y - cy) / sy) ** 2
        img = (100.0 * np.exp(-z / (2 * (1 - rho ** 2)))).astype(np.float32)
        img[0, 0] = -5.0                                          # negative pixels are clipped
        sci = np.zeros((1, 41, 41), np.float32)
        sci[0, 10:31, 10:31] = img
        _, mo = orc.coadd_stamps(sci, None, [0.0], [[20, 20]], [[0.0, 0.0]], None, R)
        w = np.maximum(img.astype(np.float64), 0)
        m00 = w.sum()
        ex, ey = np.average(X, weights=w), np.average(Y, weights=w)
        want = [m00, ex, ey, np.average((X - ex) ** 2, weights=w), np.average((Y - ey) ** 2, weights=w),
                np.average((X - ex) * (Y - ey), weights=w)]
        np.testing.assert_allclose(mo[0], want, rtol=2e-5, atol=2e-5)
        if rho == 0.0:
            np.testing.assert_allclose(mo[0, 3:5], [2.25, 2.25], rtol=1e-3)
    # an empty stamp: all zero
    _, mo = orc.coadd_stamps(np.zeros((1, 9, 9), np.float32), None, [0.0], [[4, 4]], [[0.0, 0.0]], None, 2)
    assert (mo == 0).all()


# ------------------------------------------------------------------------------------------ N5
@pytest.mark.parametrize("min_samples", [1, 3])
def test_n5_clusters_against_sklearn_dbscan(orc, min_samples):
    """scikit-learn's DBSCAN (the routine the paper used) on the scaled 4-D points: same core
    points, same partition of the core points, same noise; border points (whose cluster DBSCAN leaves
    open) must sit in a cluster with one of their core neighbours.  Coordinates on a coarse lattice,
    so no distance is within rounding of eps."""
    from sklearn.cluster import DBSCAN
    rng = np.random.default_rng(50 + min_samples)
    centres = np.stack([rng.integers(0, 400, 40), rng.integers(0, 400, 40),
                        rng.integers(-40, 40, 40) * 4, rng.integers(-40, 40, 40) * 4], 1)
    pts = np.concatenate([centres[rng.integers(0, 40, 500)] +
                          np.stack([rng.integers(-2, 3, 500), rng.integers(-2, 3, 500),
                                    rng.integers(-2, 3, 500) * 2, rng.integers(-2, 3, 500) * 2], 1),
                          np.stack([rng.integers(0, 400, 60), rng.integers(0, 400, 60),
                                    rng.integers(-160, 160, 60), rng.integers(-160, 160, 60)], 1)])
    x0y0, vxvy = pts[:, :2].astype(np.int32), pts[:, 2:].astype(np.float32)
    nu = rng.uniform(5, 50, len(pts)).astype(np.float32)
    eps_xy, eps_v = 2.5, 4.5
    label, rep = orc.cluster_candidates(x0y0, vxvy, nu, eps_xy, eps_v, min_samples)
    X = np.concatenate([x0y0 / eps_xy, vxvy.astype(np.float64) / eps_v], 1)
    ref = DBSCAN(eps=1.0, min_samples=min_samples).fit(X)
    core = np.zeros(len(pts), bool)
    core[ref.core_sample_indices_] = True
    assert ((label == -1) == (ref.labels_ == -1)).all()
    # same partition of the core points: a bijection between the two labelings
    pairs = set(zip(label[core], ref.labels_[core]))
    assert len(pairs) == len(set(label[core])) == len(set(ref.labels_[core]))
    # canonical label = smallest core index of the cluster
    for lab in set(label[core]):
        assert lab == np.flatnonzero(core & (label == lab)).min()
    d2 = ((X[:, None, :] - X[None, :, :]) ** 2).sum(-1)
    for i in np.flatnonzero(~core & (label >= 0)):            # border points
        nb = np.flatnonzero(core & (d2[i] <= 1.0))
        assert len(nb) and label[i] == label[nb].min()
    # one representative per cluster: its brightest member; every noise point is kept
    for lab in set(label[label >= 0]):
        mem = np.flatnonzero(label == lab)
        assert rep[mem].sum() == 1 and nu[mem[rep[mem] == 1][0]] == nu[mem].max()
    assert rep[label == -1].all()
    if min_samples == 3:
        assert (label == -1).any() and (~core & (label >= 0)).any(), "the case must contain noise and border points"


def test_n5_degenerate_inputs(orc):
    label, rep = orc.cluster_candidates(np.zeros((0, 2), np.int32), np.zeros((0, 2), np.float32), np.zeros(0, np.float32))
    assert len(label) == 0 and len(rep) == 0
    xy = np.array([[5, 5], [5, 5], [5, 6], [100, 100]], np.int32)
    v = np.zeros((4, 2), np.float32)
    label, rep = orc.cluster_candidates(xy, v, np.array([3.0, 3.0, 1.0, 9.0], np.float32), 1.5, 1.0, 1)
    assert list(label) == [0, 0, 0, 3] and list(rep) == [1, 0, 0, 1]       # equal nu: the smaller index wins
