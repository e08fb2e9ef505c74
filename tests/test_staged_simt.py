"""Device-side logic of the TMA-staged search kernel (csrc/search_staged.cu), run WITHOUT a GPU.

tests/hostlogic/staged_simt.cpp compiles search_staged.cu with g++ against the SIMT emulator in
tests/hostlogic/simt/ (every CUDA thread a fiber; warp collectives, __syncthreads, mbarriers with
transaction counts, tiled 3-D TMA loads with zero fill and delayed completion, bounds-checked
shared memory).  launch_search_staged then runs unchanged: host plan, tensor-map encoding, encode
kernel, and the persistent kernel with its producer warp, mbarrier ring, consumer warps,
ballot-compacted candidate queue and list insertion into the output planes.  Its six result planes
must equal the oracle's f32seq search bit for bit, for several thread schedules (forward, reverse,
pseudo-random: lanes are not in lockstep between collectives) and with TMA completions delayed.

This proves the kernel's logic (indices, barrier phases, ring and queue bookkeeping, tile
striding of the persistent CTAs); it cannot prove what only hardware decides (instruction
encodings, proxy ordering, timing).  The emulator also asserts the TMA rules it knows: 128-byte
aligned shared-memory destination and a 16-byte aligned innermost start coordinate.
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
SRC = os.path.join(HL, "staged_simt.cpp")
LIB = os.path.join(HL, "libstaged_simt.so")
CSRC = os.path.join(ROOT, "paper_1901_02492_b200", "csrc")
PLANES = ("vel_idx", "n_obs", "psi", "phi", "nu", "alpha")


@pytest.fixture(scope="module")
def sim():
    return simt_build.load("staged_simt")


def run_sim(sim, pp, times, vel, K, min_obs, order=0, seed=1, sms=3, tma_delay=0, geom=0, y_begin=0, y_end=None):
    """launch_search_staged under emulation; returns (status code, result planes, stats dict)."""
    N, H, W, _ = pp.shape
    y_end = H if y_end is None else y_end
    pp = np.ascontiguousarray(pp, np.float32)
    times = np.ascontiguousarray(times, np.float64)
    vel = np.ascontiguousarray(vel, np.float32)
    out = {k: np.full((y_end - y_begin, W, K), -77, np.int32 if k in ("vel_idx", "n_obs") else np.float32)
           for k in PLANES}
    stats = (ctypes.c_longlong * 8)()
    ptr = lambda a: a.ctypes.data_as(ctypes.c_void_p)
    rc = sim.simt_search_staged(ptr(pp), ptr(times), N, H, W, ptr(vel), int(vel.shape[0]), int(K), int(min_obs),
                                int(y_begin), int(y_end), *[ptr(out[k]) for k in PLANES], int(geom), int(order),
                                ctypes.c_uint(seed), int(sms), int(tma_delay), stats)
    names = ("smem_faults", "tma_loads", "tma_faults", "launches", "status")
    return rc, out, dict(zip(names, list(stats)))


def assert_exact(out, ref, stats, rc):
    assert rc == 0, f"launch_search_staged returned {rc}"
    assert stats["status"] == 0, "a barrier wait of the kernel timed out (pipeline logic broken)"
    assert stats["smem_faults"] == 0, "out-of-bounds or misaligned shared-memory access"
    assert stats["tma_faults"] == 0, "TMA destination or start coordinate misaligned"
    assert stats["launches"] == 2, "encode kernel + search kernel"
    for k in PLANES:
        a, b = out[k], ref[k]
        same = (a.view(np.int32) == b.view(np.int32)) | (a == b)
        assert same.all(), f"{k}: {int((~same).sum())} of {same.size} entries differ from the oracle"


def stack_case(orc, k, **over):
    cfg = synth.config(k, **over)
    st = synth.make_stack(cfg)
    pp = orc.make_psi_phi(st.sci, st.var, st.mask, st.psf)
    return cfg, st, pp


def test_config1_all_schedules(sim, orc):
    """BASELINE.json configs[0] whole, under every thread schedule and with delayed TMA completion."""
    cfg, st, pp = stack_case(orc, 1)
    ref = orc.search(pp, st.times, st.vel_grid, cfg.K, cfg.min_obs)
    loads = None
    for order, seed, sms, delay in ((0, 1, 3, 0), (1, 1, 2, 0), (2, 7, 1, 0), (2, 11, 3, 40), (0, 1, 148, 300)):
        rc, out, stats = run_sim(sim, pp, st.times, st.vel_grid, cfg.K, cfg.min_obs, order, seed, sms, delay)
        assert_exact(out, ref, stats, rc)
        assert stats["tma_loads"] > 0
        assert loads in (None, stats["tma_loads"]), "the number of boxes does not depend on the schedule"
        loads = stats["tma_loads"]
    y, x = np.unravel_index(np.argmax(out["nu"][..., 0]), out["nu"].shape[:2])
    assert (x, y) == (20, 30)


@pytest.mark.parametrize("k,over", [
    (2, dict(N=8, H=75, W=203)),                                      # odd width: padded row pitch
    (3, dict(N=15, H=70, W=133, n_sources=4)),                        # history bits, two pixels per register
    (4, dict(N=12, H=66, W=140, n_sources=4, n_angles=16, n_speeds=8)),   # K = 16: generic list insert
])
def test_crops_of_the_baseline_configs(sim, orc, k, over):
    """Crops with the full time base and velocity range: most windows leave the image, many
    trajectories have n_obs < min_obs, several tiles per persistent CTA and a ragged last tile."""
    cfg, st, pp = stack_case(orc, k, **over)
    ref = orc.search(pp, st.times, st.vel_grid, cfg.K, cfg.min_obs)
    rc, out, stats = run_sim(sim, pp, st.times, st.vel_grid, cfg.K, cfg.min_obs, order=2, seed=k, sms=2, tma_delay=25)
    assert_exact(out, ref, stats, rc)


@pytest.mark.parametrize("geom", [1, 2, 3])
def test_ring_geometries(sim, orc, geom):
    """Every ring geometry (kbmod_search_options.staged_geom): fixed slots (0 is the default of the
    other tests, 1) and the byte-granular data ring (2, 3)."""
    pp = synth.random_psiphi(9, 64, 130, seed=21, invalid_frac=0.03)
    times = np.array([0, .05, .1, .15, 1, 1.05, 1.1, 2.0, 2.05])
    vel = synth.velocity_grid(8, 6, -math.pi / 3, math.pi / 3, 3.0, 40.0)
    ref = orc.search(pp, times, vel, 8, 4)
    rc, out, stats = run_sim(sim, pp, times, vel, 8, 4, order=2, seed=geom, sms=2, tma_delay=60, geom=geom)
    assert_exact(out, ref, stats, rc)


def test_interior_trajectories_fill_the_lists(sim, orc):
    """Slow velocities: every trajectory is eligible, the queue overflows 32 inside a block (batch
    flush in the middle of the scoring switch) and same-pixel candidates meet in one batch."""
    pp = synth.random_psiphi(6, 60, 128, seed=5, invalid_frac=0.02)
    times = np.array([0, .1, .2, 1.0, 1.1, 1.2])
    vel = synth.velocity_grid(10, 8, -math.pi, math.pi, 0.5, 6.0)
    for K, mo in ((8, 2), (3, 6), (32, 1)):
        ref = orc.search(pp, times, vel, K, mo)
        rc, out, stats = run_sim(sim, pp, times, vel, K, mo, order=2, seed=K, sms=3, tma_delay=10)
        assert_exact(out, ref, stats, rc)


def test_unproven_shifts_take_the_literal_path(sim, orc):
    """Exact-half and near-half v*dt: ENT_UNSAFE entries run S3 per lane on the device."""
    H, W = 31, 200
    pp = np.zeros((3, H, W, 2), np.float32)
    pp[1:, ..., 0] = (np.arange(H)[:, None] * W + np.arange(W)[None, :]).astype(np.float32)[None]
    pp[0, ..., 0] = 0.25
    pp[..., 1] = 1.0
    times = np.array([0.0, 0.5, 1.0])
    vel = np.array([[3.0, 1.0], [-3.0, -1.0], [1.0, 3.0], [10.49999, 0.0], [20.99998, 0.5],
                    [0.49999997, 0.49999997], [0.99999994, -0.99999994], [7.0, 7.0],
                    [-0.5, 0.0], [99.5, 0.0], [199.0, 1.0], [10.5, 10.5]], np.float32)
    ref = orc.search(pp, times, vel, 4, 2)
    rc, out, stats = run_sim(sim, pp, times, vel, 4, 2, order=1, sms=2)
    assert_exact(out, ref, stats, rc)


def test_degenerate_shapes(sim, orc):
    # N = 1: no image to shift (one NOP entry per block, no TMA at all)
    pp = synth.random_psiphi(1, 1, 33, seed=1, invalid_frac=0.2)
    vel0 = np.zeros((1, 2), np.float32)
    rc, out, stats = run_sim(sim, pp, [3.0], vel0, 2, 1)
    assert_exact(out, orc.search(pp, [3.0], vel0, 2, 1), stats, rc)
    assert stats["tma_loads"] == 0
    # velocities far beyond the image, unsorted times, duplicated velocities, V not a multiple of 8
    pp = synth.random_psiphi(5, 37, 70, seed=3, invalid_frac=0.1)
    vel = synth.velocity_grid(4, 4, -2, 2, 2, 12)
    vel = np.concatenate([vel, vel[3:9], vel[:2], np.array([[5e4, 0], [0, -7e4], [3e3, 3e3]], np.float32)])
    times = np.array([5.0, 4.5, 6.0, 5.25, 7.0])
    ref = orc.search(pp, times, vel, 8, 3)
    rc, out, stats = run_sim(sim, pp, times, vel, 8, 3, order=2, seed=3, sms=5, tma_delay=15)
    assert_exact(out, ref, stats, rc)
    # everything invalid: only sentinels
    pp = synth.random_psiphi(4, 10, 40, seed=2, invalid_frac=1.0)
    ref = orc.search(pp, np.arange(4.0), vel[:9], 4, 1)
    rc, out, stats = run_sim(sim, pp, np.arange(4.0), vel[:9], 4, 1)
    assert_exact(out, ref, stats, rc)
    assert (out["vel_idx"] == -1).all()


def test_limit_cases(sim, orc):
    """Image sizes around the 64 x 30 tile (one short, exact, one over; one row, one column) and
    shifts at the edge of the int16 encoding (|v*dt| around SH_LIMIT = 30000, both signs)."""
    vel = synth.velocity_grid(3, 3, -math.pi, math.pi, 1.0, 30.0)
    for H, W in ((29, 63), (30, 64), (31, 65), (1, 129), (61, 1), (60, 128)):
        pp = synth.random_psiphi(4, H, W, seed=H * 1000 + W, invalid_frac=0.1)
        times = np.array([0.0, 0.4, 1.0, 1.7])
        rc, out, stats = run_sim(sim, pp, times, vel, 4, 2, order=2, seed=H, sms=2, tma_delay=7)
        assert_exact(out, orc.search(pp, times, vel, 4, 2), stats, rc)
    pp = synth.random_psiphi(3, 40, 70, seed=9, invalid_frac=0.0)
    big = np.array([[29999.4, 0.0], [-29999.4, 0.0], [0.0, 29999.4], [0.0, -29999.4], [30000.5, 0.0],
                    [-30000.5, 29999.4], [29999.6, -29999.6], [30000.4, 30000.4], [1.0, 1.0], [15999.7, -15999.7],
                    [3e38, 0.0], [-3e38, -3e38]], np.float32)
    times = np.array([0.0, 1.0, 2.0])
    rc, out, stats = run_sim(sim, pp, times, big, 4, 1, order=1, sms=3)
    assert_exact(out, orc.search(pp, times, big, 4, 1), stats, rc)


def test_row_bands_equal_the_full_search(sim, orc):
    """kbmod_search_rows on the staged kernel: bands (tile-aligned or not, one row, empty, the last
    rows) equal the same rows of the oracle's full search; the planes hold the band only."""
    pp = synth.random_psiphi(5, 70, 90, seed=31, invalid_frac=0.1)
    times = np.array([0.0, 0.3, 1.0, 1.4, 2.0])
    vel = synth.velocity_grid(4, 3, -math.pi, math.pi, 1.0, 20.0)
    full = orc.search(pp, times, vel, 4, 2)
    for y0, y1 in ((0, 30), (30, 70), (5, 41), (69, 70), (17, 17), (0, 70)):
        rc, out, stats = run_sim(sim, pp, times, vel, 4, 2, order=2, seed=y0 + 1, sms=2, tma_delay=9, y_begin=y0, y_end=y1)
        if y1 == y0:
            stats["launches"] += 1            # an empty band launches the encode kernel only
        assert_exact(out, {k: v[y0:y1] for k, v in full.items()}, stats, rc)


def test_image_count_variants(sim, orc):
    """N = 20 (one history register per pixel), N = 40 and N = 64 = KBMOD_MAX_IMAGES (additive counts)."""
    rng = np.random.default_rng(64)
    for N, mo in ((20, 9), (40, 20), (64, 20)):
        pp = synth.random_psiphi(N, 32, 70, seed=N, invalid_frac=0.05)
        times = np.sort(rng.uniform(0.0, 5.0, N))
        vel = synth.velocity_grid(6, 4, -math.pi / 2, math.pi / 2, 1.0, 9.0)
        ref = orc.search(pp, times, vel, 8, mo)
        rc, out, stats = run_sim(sim, pp, times, vel, 8, mo, order=2, seed=N, sms=2, tma_delay=20)
        assert_exact(out, ref, stats, rc)


@pytest.mark.parametrize("geom", [0, 3])
def test_randomized_shapes(sim, orc, geom):
    """25 seeded random problems per ring kind, random schedule, CTA count and TMA delay (a longer
    run of the same generator, 2 025 cases on a fixed and a variable ring, found no mismatch)."""
    from tests.test_tiled_simt import random_case
    rng = np.random.default_rng(77 + geom)
    for _ in range(25):
        pp, times, vel, K, mo = random_case(rng)
        rc, out, stats = run_sim(sim, pp, times, vel, K, mo, int(rng.integers(3)), int(rng.integers(1 << 30)),
                                 int(rng.integers(1, 5)), int(rng.choice([0, 10, 100])), geom=geom)
        assert_exact(out, orc.search(pp, times, vel, K, mo), stats, rc)
