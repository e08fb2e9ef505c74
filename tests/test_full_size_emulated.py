"""BASELINE.json configs AT FULL SIZE under the SIMT emulator (opt-in: KBMOD_TEST_FULL_SIZE_EMULATED=1;
tens of minutes and about 10 GB of host memory, so not part of the default CPU suite).

The product's launch code and search kernels (compiled with g++ against tests/hostlogic/simt/) search
BANDS of start rows of a full-size stack with the full velocity grid through the row-band call -- the
top edge, a tile seam in the interior (where every window of most velocity blocks lies inside the
image: the branch-free paths with the real, up to 1 560 px shifts and element offsets near 2^28) and
the bottom edge -- and every result plane must equal the oracle's bit for bit.  This is the closest a
machine without a GPU gets to the full-size parity tests of tests/test_gpu_parity.py; it says
nothing about hardware.  When it was last run, and what it showed: DESIGN.md section 8.
"""
import os
import time

import numpy as np
import pytest

from paper_1901_02492_b200 import synth
from tests import simt_build, test_staged_simt as S, test_tiled_simt as T

pytestmark = pytest.mark.skipif(os.environ.get("KBMOD_TEST_FULL_SIZE_EMULATED") != "1",
                                reason="opt-in: KBMOD_TEST_FULL_SIZE_EMULATED=1 (tens of minutes)")
BANDS = ((0, 32), (2040, 2072), (4080, 4096))


def _grid(cfg):
    times = synth.make_times(cfg, np.random.default_rng(cfg.seed))
    vel = synth.velocity_grid(cfg.n_angles, cfg.n_speeds, cfg.ang_lo, cfg.ang_hi, cfg.speed_lo, cfg.speed_hi)
    return times, vel


@pytest.fixture(scope="module")
def stack():
    """BASELINE.json configs[2]: 15 x 4096 x 4096, 32 x 20 velocities, K = 8, min_obs = 8."""
    cfg = synth.config(3)
    times, vel = _grid(cfg)
    pp = synth.random_psiphi(cfg.N, cfg.H, cfg.W, seed=33, invalid_frac=0.01)      # 2 GB; the search does not care
    return cfg, times, vel, pp


@pytest.fixture(scope="module")
def reference(stack, orc):
    cfg, times, vel, pp = stack
    return {b: orc.search(pp, times, vel, cfg.K, cfg.min_obs, y_begin=b[0], y_end=b[1]) for b in BANDS}


@pytest.mark.parametrize("kernel", ["tiled", "queued", "staged"])
def test_bands_of_the_full_size_stack(stack, reference, kernel):
    cfg, times, vel, pp = stack
    for (y0, y1) in BANDS:
        t = time.time()
        if kernel == "staged":
            rc, out, stats = S.run_sim(simt_build.load("staged_simt"), pp, times, vel, cfg.K, cfg.min_obs, order=0,
                                       sms=8, y_begin=y0, y_end=y1)
            S.assert_exact(out, reference[(y0, y1)], stats, rc)
        else:
            out = T.run_sim(simt_build.load("tiled_simt"), pp, times, vel, cfg.K, cfg.min_obs,
                            T.QUEUED if kernel == "queued" else T.TILED, order=0, y_begin=y0, y_end=y1)
            T.assert_exact(out, reference[(y0, y1)])
        print(f"config3 {kernel} rows [{y0}, {y1}): bit-exact, {time.time() - t:.0f} s", flush=True)


@pytest.mark.parametrize("name,k,over,bands", [
    # BASELINE.json configs[1]: 8 x 2048 x 4096 (H < W), V = 512
    ("config2", 2, {}, ((0, 32), (1016, 1048), (2040, 2048))),
    # BASELINE.json configs[3]: K = 16 (64 x 16 tiles, blocks of 16), V = 2048, irregular times, N = 12
    ("config4", 4, {}, ((0, 16), (2048, 2064), (4088, 4096))),
    # configs[4], the far corners of the sweep: N = 40 (additive counters, 5.4 GB stack) and V = 8192
    ("config5_N40", 5, dict(N=40), ((2040, 2056),)),
    ("config5_V8192", 5, dict(N=10, n_angles=128, n_speeds=64), ((0, 8), (4088, 4096))),
])
@pytest.mark.parametrize("kernel", ["tiled", "queued"])
def test_bands_of_the_other_full_size_configs(orc, name, k, over, bands, kernel):
    cfg = synth.config(k, **over)
    times, vel = _grid(cfg)
    pp = synth.random_psiphi(cfg.N, cfg.H, cfg.W, seed=40 + k, invalid_frac=0.1 if k == 4 else 0.01)
    for (y0, y1) in bands:
        t = time.time()
        ref = orc.search(pp, times, vel, cfg.K, cfg.min_obs, y_begin=y0, y_end=y1)
        out = T.run_sim(simt_build.load("tiled_simt"), pp, times, vel, cfg.K, cfg.min_obs,
                        T.QUEUED if kernel == "queued" else T.TILED, order=0, y_begin=y0, y_end=y1)
        T.assert_exact(out, ref)
        print(f"{name} {kernel} rows [{y0}, {y1}): bit-exact, {time.time() - t:.0f} s", flush=True)


def test_staged_kernel_band_of_config4(orc):
    """Kernel 3 at BASELINE.json configs[3]: K = 16 (generic list insert), V = 2048, irregular times."""
    cfg = synth.config(4)
    times, vel = _grid(cfg)
    pp = synth.random_psiphi(cfg.N, cfg.H, cfg.W, seed=44, invalid_frac=0.1)
    y0, y1 = 2040, 2070                                   # one 30-row tile row in the interior
    t = time.time()
    ref = orc.search(pp, times, vel, cfg.K, cfg.min_obs, y_begin=y0, y_end=y1)
    rc, out, stats = S.run_sim(simt_build.load("staged_simt"), pp, times, vel, cfg.K, cfg.min_obs, order=0, sms=8,
                               y_begin=y0, y_end=y1)
    S.assert_exact(out, ref, stats, rc)
    print(f"config4 staged rows [{y0}, {y1}): bit-exact, {time.time() - t:.0f} s", flush=True)


def test_psi_phi_on_full_size_images(orc):
    """kbmod_make_psi_phi's one-launch kernel on two full 4096 x 4096 images of configs[2] (P = 21;
    8 192 tiles per image, the image index decoded from blockIdx.x): bands of rows at the top edge, at
    a tile seam and at the bottom edge against the oracle run on the same rows plus the PSF halo."""
    import ctypes
    from tests.test_post_simt import assert_psiphi_close, run_psi_phi
    cfg = synth.config(3, N=2, n_sources=50)
    st = synth.make_stack(cfg)
    t = time.time()
    got, launches = run_psi_phi(simt_build.load("post_simt"), st.sci, st.var, st.mask, st.psf)
    assert launches == 1
    print(f"psi/phi of 2 x 4096 x 4096 emulated in {time.time() - t:.0f} s", flush=True)
    r = (st.psf.shape[-1] - 1) // 2
    for y0 in (0, 28, 2044, cfg.H - 8):
        a, b = max(0, y0 - r), min(cfg.H, y0 + 8 + r)
        ref, pabs = orc.make_psi_phi(st.sci[:, a:b], st.var[:, a:b], st.mask[:, a:b], st.psf, want_abs=True)
        sl = slice(y0 - a, y0 - a + 8)
        assert_psiphi_close(got[:, y0:y0 + 8], ref[:, sl], pabs[:, sl])
    assert np.isnan(got[..., 0]).mean() > 0.005          # the 1 % mask is there
