"""Device-side logic of the tiled search kernels (csrc/search_tiled.cu), run WITHOUT a GPU under
the SIMT emulator of tests/hostlogic/simt/ (see tests/test_staged_simt.py for what it models).

* search_tiled_kernel (kernel id 2, the default path) is validated bit for bit on B200 hardware
  (tests/test_gpu_parity.py); reproducing the oracle here as well checks the EMULATOR.
* search_tiledq_kernel (kernel id 4: the same gathers, survivors of the pre-test compacted into
  per-warp queues, lists in the output planes) must equal the oracle's f32seq search bit for bit
  for several thread schedules (lanes are not in lockstep between warp collectives).
"""
import ctypes
import math
import os
import subprocess

import numpy as np
import pytest

from paper_1901_02492_b200 import synth
from tests import simt_build

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
HL = os.path.join(ROOT, "tests", "hostlogic")
SRC = os.path.join(HL, "tiled_simt.cpp")
LIB = os.path.join(HL, "libtiled_simt.so")
CSRC = os.path.join(ROOT, "paper_1901_02492_b200", "csrc")
PLANES = ("vel_idx", "n_obs", "psi", "phi", "nu", "alpha")
TILED, QUEUED = 0, 1


@pytest.fixture(scope="module")
def sim():
    return simt_build.load("tiled_simt")


def run_sim(sim, pp, times, vel, K, min_obs, queued, order=0, seed=1, y_begin=0, y_end=None, group_w=0):
    N, H, W, _ = pp.shape
    y_end = H if y_end is None else y_end
    pp = np.ascontiguousarray(pp, np.float32)
    times = np.ascontiguousarray(times, np.float64)
    vel = np.ascontiguousarray(vel, np.float32)
    out = {k: np.full((y_end - y_begin, W, K), -77, np.int32 if k in ("vel_idx", "n_obs") else np.float32)
           for k in PLANES}
    stats = (ctypes.c_longlong * 8)()
    ptr = lambda a: a.ctypes.data_as(ctypes.c_void_p)
    rc = sim.simt_search_tiled(ptr(pp), ptr(times), N, H, W, ptr(vel), int(vel.shape[0]), int(K), int(min_obs),
                               int(y_begin), int(y_end), *[ptr(out[k]) for k in PLANES], int(queued), int(group_w),
                               int(order), ctypes.c_uint(seed), stats)
    assert rc == 0, f"launch_search_tiled returned {rc}"
    assert stats[3] == (2 if y_end > y_begin else 1), "encode kernel + search kernel"
    return out


def assert_exact(out, ref):
    for k in PLANES:
        a, b = out[k], ref[k]
        same = (a.view(np.int32) == b.view(np.int32)) | (a == b)
        assert same.all(), f"{k}: {int((~same).sum())} of {same.size} entries differ from the oracle"


def stack_case(orc, k, **over):
    cfg = synth.config(k, **over)
    st = synth.make_stack(cfg)
    return cfg, st, orc.make_psi_phi(st.sci, st.var, st.mask, st.psf)


@pytest.mark.parametrize("queued", [TILED, QUEUED])
def test_config1(sim, orc, queued):
    cfg, st, pp = stack_case(orc, 1)
    ref = orc.search(pp, st.times, st.vel_grid, cfg.K, cfg.min_obs)
    for order, seed in ((0, 1), (1, 1), (2, 9)):
        out = run_sim(sim, pp, st.times, st.vel_grid, cfg.K, cfg.min_obs, queued, order, seed)
        assert_exact(out, ref)
    y, x = np.unravel_index(np.argmax(out["nu"][..., 0]), out["nu"].shape[:2])
    assert (x, y) == (20, 30)


@pytest.mark.parametrize("queued", [TILED, QUEUED])
@pytest.mark.parametrize("k,over", [
    (2, dict(N=8, H=75, W=203)),                                      # odd width, ragged tiles
    (3, dict(N=15, H=70, W=133, n_sources=4)),
    (4, dict(N=12, H=66, W=140, n_sources=4, n_angles=16, n_speeds=8)),   # K = 16: blocks of 16, generic insert
])
def test_crops_of_the_baseline_configs(sim, orc, queued, k, over):
    cfg, st, pp = stack_case(orc, k, **over)
    ref = orc.search(pp, st.times, st.vel_grid, cfg.K, cfg.min_obs)
    assert_exact(run_sim(sim, pp, st.times, st.vel_grid, cfg.K, cfg.min_obs, queued, order=2, seed=k), ref)


def test_queued_interior_trajectories_fill_the_lists(sim, orc):
    """Slow velocities keep every window inside the image (the fast path of the gathers) and make
    every trajectory eligible: queues overflow 32 inside a block, same-pixel candidates meet in
    one batch; K = 3 / 8 (register insert), 16 and 32 (generic insert, other tile shapes)."""
    pp = synth.random_psiphi(6, 100, 140, seed=5, invalid_frac=0.02)    # tiles (1,1), (1,2): all windows inside
    times = np.array([0, .1, .2, 1.0, 1.1, 1.2])
    vel = synth.velocity_grid(10, 8, -math.pi, math.pi, 0.5, 6.0)
    for K, mo, order in ((8, 2, 2), (3, 6, 1), (16, 1, 2), (32, 1, 0)):
        ref = orc.search(pp, times, vel, K, mo)
        assert_exact(run_sim(sim, pp, times, vel, K, mo, QUEUED, order, seed=K), ref)


def test_queued_unproven_shifts_and_degenerate_shapes(sim, orc):
    H, W = 31, 200
    pp = np.zeros((3, H, W, 2), np.float32)
    pp[1:, ..., 0] = (np.arange(H)[:, None] * W + np.arange(W)[None, :]).astype(np.float32)[None]
    pp[0, ..., 0] = 0.25
    pp[..., 1] = 1.0
    times = np.array([0.0, 0.5, 1.0])
    vel = np.array([[3.0, 1.0], [-3.0, -1.0], [1.0, 3.0], [10.49999, 0.0], [20.99998, 0.5],
                    [0.49999997, 0.49999997], [0.99999994, -0.99999994], [7.0, 7.0],
                    [-0.5, 0.0], [99.5, 0.0], [199.0, 1.0], [10.5, 10.5]], np.float32)
    assert_exact(run_sim(sim, pp, times, vel, 4, 2, QUEUED, order=1), orc.search(pp, times, vel, 4, 2))
    # N = 1
    pp = synth.random_psiphi(1, 1, 33, seed=1, invalid_frac=0.2)
    vel0 = np.zeros((1, 2), np.float32)
    assert_exact(run_sim(sim, pp, [3.0], vel0, 2, 1, QUEUED), orc.search(pp, [3.0], vel0, 2, 1))
    # far velocities, unsorted times, duplicated velocities, V not a multiple of the block
    pp = synth.random_psiphi(5, 37, 70, seed=3, invalid_frac=0.1)
    vel = synth.velocity_grid(4, 4, -2, 2, 2, 12)
    vel = np.concatenate([vel, vel[3:9], vel[:2], np.array([[5e4, 0], [0, -7e4], [3e3, 3e3]], np.float32)])
    times = np.array([5.0, 4.5, 6.0, 5.25, 7.0])
    assert_exact(run_sim(sim, pp, times, vel, 8, 3, QUEUED, order=2, seed=3), orc.search(pp, times, vel, 8, 3))
    # everything invalid: only sentinels
    pp = synth.random_psiphi(4, 10, 40, seed=2, invalid_frac=1.0)
    out = run_sim(sim, pp, np.arange(4.0), vel[:9], 4, 1, QUEUED)
    assert_exact(out, orc.search(pp, np.arange(4.0), vel[:9], 4, 1))
    assert (out["vel_idx"] == -1).all()


def test_queued_image_count_variants(sim, orc):
    """N = 16 (the largest stack counted with history bits), 17 and above (additive counters),
    N = 64 = KBMOD_MAX_IMAGES; slow velocities and a 100 x 140 image so interior tiles take the
    branch-free path in both counting modes."""
    rng = np.random.default_rng(64)
    for N, mo in ((16, 16), (17, 9), (40, 20), (64, 20)):
        pp = synth.random_psiphi(N, 100 if N < 20 else 34, 140 if N < 20 else 70, seed=N, invalid_frac=0.05)
        times = np.sort(rng.uniform(0.0, 5.0, N))
        vel = synth.velocity_grid(6, 4, -math.pi / 2, math.pi / 2, 1.0, 9.0)
        assert_exact(run_sim(sim, pp, times, vel, 8, mo, QUEUED, order=2, seed=N), orc.search(pp, times, vel, 8, mo))


@pytest.mark.parametrize("queued", [TILED, QUEUED])
def test_limit_cases(sim, orc, queued):
    """The limits the GPU tests do not reach: image sizes around the 64 x 32 tile (one short, exact,
    one over; one row, one column), shifts at the edge of the int16 shift encoding (|v*dt| around
    SH_LIMIT = 32000: proven, skipped, and both signs), and blocks whose clean velocities are
    completed with benign padding while the tile touches every image corner."""
    rng = np.random.default_rng(5)
    vel = synth.velocity_grid(3, 3, -math.pi, math.pi, 1.0, 30.0)
    for H, W in ((31, 63), (32, 64), (33, 65), (1, 129), (70, 1), (64, 128)):
        pp = synth.random_psiphi(4, H, W, seed=H * 1000 + W, invalid_frac=0.1)
        times = np.array([0.0, 0.4, 1.0, 1.7])
        assert_exact(run_sim(sim, pp, times, vel, 4, 2, queued, order=2, seed=H), orc.search(pp, times, vel, 4, 2))
    # shifts at the limits of the encoding: +-31999.4 is a proven shift, 32000.5 is skipped; the image
    # is tiny, so every such window is far outside (no sample may be fetched, n_obs counts image 0 only)
    pp = synth.random_psiphi(3, 40, 70, seed=9, invalid_frac=0.0)
    big = np.array([[31999.4, 0.0], [-31999.4, 0.0], [0.0, 31999.4], [0.0, -31999.4], [32000.5, 0.0],
                    [-32000.5, 31999.4], [29999.6, -29999.6], [30000.4, 30000.4], [1.0, 1.0], [15999.7, -15999.7],
                    [3e38, 0.0], [-3e38, -3e38]], np.float32)
    times = np.array([0.0, 1.0, 2.0])
    assert_exact(run_sim(sim, pp, times, big, 4, 1, queued, order=1), orc.search(pp, times, big, 4, 1))
    # half-integer velocities inside chunks of clean ones (kernel 4: benign padding next to the corners)
    vel = synth.velocity_grid(4, 5, -math.pi, math.pi, 2.0, 24.0)
    vel[[1, 6, 7, 13]] = np.array([[10.5, 3.0], [-2.5, -7.5], [0.5, 0.5], [63.5, 31.5]], np.float32)
    pp = synth.random_psiphi(5, 33, 66, seed=12, invalid_frac=0.2)
    times = np.array([0.0, 1.0, 2.0, 3.0, 1.0])
    assert_exact(run_sim(sim, pp, times, vel, 8, 2, queued, order=2, seed=3), orc.search(pp, times, vel, 8, 2))


def test_limit_on_stack_size_is_refused_before_any_access(sim):
    """(N+1)*H*W + SH_LIMIT*(W+1) must stay below 2^31 (int32 element offsets): the launch returns
    KBMOD_ERR_UNSUPPORTED (-6) without touching a buffer (all pointers are NULL here)."""
    assert sim.simt_tiled_limits(15, 11000, 11000, 8, 8) == -6        # 16 * 1.21e8 = 1.9e9 + 3.5e8 > 2^31
    assert sim.simt_tiled_limits(3, 30001, 100, 8, 8) == -6           # beyond the int16 shift range
    assert sim.simt_tiled_limits(64, 8192, 8192, 8, 8) == -6          # 65 * 2^26 > 2^31


def random_case(rng):
    """One random small search problem: shapes, K, min_obs, grids with exact halves, unsorted times,
    heavy masking, images with few distinct values (many exact nu ties)."""
    N = int(rng.choice([1, 2, 3, 5, 8, 12, 15, 16, 17, 24, 33]))
    H, W = int(rng.integers(1, 100)), int(rng.integers(1, 200))
    K, mo = int(rng.choice([1, 2, 4, 8, 9, 16, 32])), int(rng.integers(1, N + 1))
    vel = synth.velocity_grid(int(rng.integers(1, 7)), int(rng.integers(1, 7)), -math.pi * rng.random(),
                              math.pi * rng.random(), 0.0 if rng.random() < 0.3 else 0.5,
                              float(rng.choice([2.0, 10.0, 60.0, 400.0])))
    if rng.random() < 0.3:
        vel = (np.round(vel * 2) / 2).astype(np.float32)
    times = np.sort(rng.uniform(0, 3, N)) if rng.random() < 0.7 else rng.uniform(0, 3, N)
    if rng.random() < 0.3:
        times = np.round(times * 2) / 2
    pp = synth.random_psiphi(N, H, W, seed=int(rng.integers(1 << 30)), invalid_frac=float(rng.choice([0.0, 0.05, 0.5])))
    if rng.random() < 0.3:
        pp[..., 0] = np.where(np.isnan(pp[..., 0]), np.nan, np.round(pp[..., 0]))
        pp[..., 1] = np.where(np.isnan(pp[..., 0]), 0, 1.0)
    return pp, times, vel.astype(np.float32), K, mo


def test_queued_randomized_shapes(sim, orc):
    """40 seeded random problems (a longer run of the same generator, 2 875 cases, found no
    mismatch when kernel 4 was written)."""
    rng = np.random.default_rng(2024)
    for _ in range(40):
        pp, times, vel, K, mo = random_case(rng)
        out = run_sim(sim, pp, times, vel, K, mo, QUEUED, int(rng.integers(3)), int(rng.integers(1 << 30)))
        assert_exact(out, orc.search(pp, times, vel, K, mo))


@pytest.mark.parametrize("gw", [1, 3, 200])
def test_queued_tile_order_knob_does_not_change_results(sim, orc, gw):
    """kbmod_search_options.tile_group_w only permutes which CTA takes which tile."""
    cfg, st, pp = stack_case(orc, 3, N=15, H=70, W=300, n_sources=4)        # 5 x 3 tiles, ragged on both axes
    ref = orc.search(pp, st.times, st.vel_grid, cfg.K, cfg.min_obs)
    assert_exact(run_sim(sim, pp, st.times, st.vel_grid, cfg.K, cfg.min_obs, QUEUED, order=2, seed=gw, group_w=gw), ref)


@pytest.mark.parametrize("queued", [TILED, QUEUED])
def test_row_bands_equal_the_full_search(sim, orc, queued):
    """kbmod_search_rows: bands of start rows (tile-aligned or not, one row, empty, the last rows)
    equal the same rows of the oracle's full search; the planes hold the band only."""
    pp = synth.random_psiphi(5, 70, 90, seed=31, invalid_frac=0.1)
    times = np.array([0.0, 0.3, 1.0, 1.4, 2.0])
    vel = synth.velocity_grid(4, 3, -math.pi, math.pi, 1.0, 20.0)
    full = orc.search(pp, times, vel, 4, 2)
    for y0, y1 in ((0, 32), (32, 70), (5, 41), (69, 70), (17, 17), (0, 70)):
        out = run_sim(sim, pp, times, vel, 4, 2, queued, order=2, seed=y0 + 1, y_begin=y0, y_end=y1)
        assert_exact(out, {k: v[y0:y1] for k, v in full.items()})
