"""Host logic of the TMA-staged search kernel, checked without a GPU.

kbmod_debug_staged_plan returns the entry stream the kernel executes.  This test interprets the
stream in NumPy exactly as the device code in csrc/search_staged.cu does -- boxes copied from
the (psi, -phi) encoded stack with zero fill outside the image, one window per member read at
`member offset + row * pitch`, fp32 adds in entry order, validity = sign bit of the second word,
literal positions for the entries whose shift the host could not prove -- and compares the
resulting Psi / Phi / n_obs of EVERY (start pixel, velocity) with the oracle's dense evaluation,
bit for bit.  A wrong shift proof, a wrong box origin or member offset, a velocity that is
missing or visited twice, or images out of order would all show up here.
"""
import math

import numpy as np
import pytest

from paper_1901_02492_b200 import binding, synth

ENT_NOP, ENT_TMA, ENT_UNSAFE = 0, 1, 2
FLAG_LAST = 1


def encode(pp):
    """(psi, phi) -> (psi, -phi), invalid -> (+0, +0), row pitch padded to even (zero column)."""
    N, H, W, _ = pp.shape
    Wp = (W + 1) & ~1
    enc = np.zeros((N, H, Wp, 2), np.float32)
    ok = ~np.isnan(pp[..., 0])
    enc[:, :, :W, 0] = np.where(ok, pp[..., 0], np.float32(0))
    enc[:, :, :W, 1] = np.where(ok, -pp[..., 1], np.float32(0))
    return enc


def fetch_box(enc, img, gx, gy, bw, bh):
    """TMA tile load with zero fill: box[y, x] = enc[img, gy + y, gx + x] or 0 outside."""
    N, H, Wp, _ = enc.shape
    box = np.zeros((bh, bw, 2), np.float32)
    y0, y1 = max(gy, 0), min(gy + bh, H)
    x0, x1 = max(gx, 0), min(gx + bw, Wp)
    if y0 < y1 and x0 < x1:
        box[y0 - gy:y1 - gy, x0 - gx:x1 - gx] = enc[img, y0:y1, x0:x1]
    return box


def literal_pixels(p0, v, dt, n):
    """S3 as include/kbmod_b200.h states it, in float32 (NumPy keeps each operation in binary32)."""
    f = p0.astype(np.float32) + np.float32(np.float32(v) * np.float32(dt))
    g = np.floor(f + np.float32(0.5))
    ok = (g >= 0) & (g < n)
    return np.where(ok, g, 0).astype(np.int64), ok


def run_plan(pp, times, vel, tiles=None, geom=0):
    """Interprets the plan for the given tiles; returns dict (tile_x, tile_y) -> Psi, Phi, n of
    shape [TH, TW, V] (only pixels inside the image are meaningful)."""
    N, H, W, _ = pp.shape
    stream, shapes, info = binding.debug_staged_plan(times, N, H, W, vel, geom)
    TW, TH, B = info["TW"], info["TH"], info["B"]
    enc = encode(pp)
    dt = (np.asarray(times, np.float64) - float(times[0])).astype(np.float32)
    V = vel.shape[0]
    tiles_x, tiles_y = -(-W // TW), -(-H // TH)
    if tiles is None:
        tiles = [(tx, ty) for ty in range(tiles_y) for tx in range(tiles_x)]
    seen = np.zeros(V, np.int64)
    out = {}
    for (tx, ty) in tiles:
        tile_x, tile_y = tx * TW, ty * TH
        py, px = np.meshgrid(np.arange(TH), np.arange(TW), indexing="ij")
        # image 0: shift (0, 0); pixels outside the image contribute the zero sample
        s0 = fetch_box(enc, 0, tile_x, tile_y, TW, TH)
        s0[(tile_y + py >= H) | (tile_x + px >= W)] = 0
        Psi = np.zeros((TH, TW, V), np.float32)
        Phi = np.zeros((TH, TW, V), np.float32)
        cnt = np.zeros((TH, TW, V), np.int32)
        acc = None
        for e in stream:
            if acc is None:            # a block starts
                acc = np.repeat(s0[None], B, 0).copy()
                n = np.repeat(np.signbit(s0[..., 1])[None].astype(np.int32), B, 0)
            typ, flags, img = e[0] & 0xFF, (e[0] >> 8) & 0xFF, e[0] >> 16
            if typ == ENT_TMA:
                ox = int(np.int16(e[3] & 0xFFFF))
                oy = int(e[3] >> 16)
                bw, bh = int(e[4] & 0xFFFF), int(e[4] >> 16)
                assert tuple(shapes[e[5]]) == (bw, bh) and e[2] == bw * 8
                assert (tile_x + ox) % 2 == 0, "TMA box start must be 16-byte aligned"
                assert bw % 2 == 0 and bw * bh <= info["CAP"] and 2 * bw <= 256 and bh <= 256
                box = fetch_box(enc, img, tile_x + ox, tile_y + oy, bw, bh).reshape(-1, 2)
                for b in range(B):
                    if e[1] >> b & 1:
                        off = e[8 + b]                         # bytes from the box start
                        assert off >= 0 and off % 8 == 0
                        idx = off // 8 + py * bw + px          # thread address: + row*pitch + x*8
                        assert idx.max() < bw * bh, "window leaves the box"
                        s = box[idx]
                        acc[b] = acc[b] + s                    # fp32, one add per image in order
                        n[b] += np.signbit(s[..., 1])
            elif typ == ENT_UNSAFE:
                b = int(e[5])
                vx, vy = np.array(e[6:8], np.int32).view(np.float32)
                ix, okx = literal_pixels(tile_x + px, vx, dt[img], W)
                iy, oky = literal_pixels(tile_y + py, vy, dt[img], H)
                s = np.where((okx & oky)[..., None], enc[img, iy, ix], np.float32(0))
                acc[b] = acc[b] + s
                n[b] += np.signbit(s[..., 1])
            if flags & FLAG_LAST:
                for b in range(B):
                    j = e[8 + B + b]
                    if j >= 0:
                        seen[j] += 1
                        Psi[..., j], Phi[..., j], cnt[..., j] = acc[b, ..., 0], -acc[b, ..., 1], n[b]
                acc = None
        assert acc is None, "stream must end on a FLAG_LAST entry"
        out[(tile_x, tile_y)] = (Psi, Phi, cnt)
    assert (seen == len(tiles)).all(), "every velocity exactly once per tile"
    return out, info


def check_against_oracle(orc, pp, times, vel, tiles=None, geom=0):
    N, H, W, _ = pp.shape
    res, info = run_plan(pp, times, vel, tiles, geom)
    rPsi, rPhi, rn = orc.eval_all(pp, times, vel)           # [H, W, V], f32seq
    for (tile_x, tile_y), (Psi, Phi, cnt) in res.items():
        h, w = min(info["TH"], H - tile_y), min(info["TW"], W - tile_x)
        sl = (slice(tile_y, tile_y + h), slice(tile_x, tile_x + w))
        assert (cnt[:h, :w] == rn[sl]).all()
        assert (Psi[:h, :w].view(np.int32) == rPsi[sl].view(np.int32)).all() or (Psi[:h, :w] == rPsi[sl]).all()
        assert (Phi[:h, :w] == rPhi[sl]).all()


@pytest.mark.parametrize("k,over", [
    (1, {}),
    (2, dict(N=8, H=75, W=203)),
    (3, dict(N=15, H=70, W=133, n_sources=4)),
    (4, dict(N=12, H=66, W=140, n_sources=4, n_angles=16, n_speeds=8)),
])
def test_plan_reproduces_oracle_on_crops(orc, k, over):
    cfg = synth.config(k, **over)
    st = synth.make_stack(cfg)
    pp = orc.make_psi_phi(st.sci, st.var, st.mask, st.psf)
    check_against_oracle(orc, pp, st.times, st.vel_grid)


@pytest.mark.parametrize("geom", [1, 2, 3])
def test_plan_ring_geometry_variants(orc, geom):
    """kbmod_search_options.staged_geom selects other slot sizes: the plan must stay exact and
    respect the cap."""
    cfg = synth.config(3, N=15, H=70, W=133, n_sources=4)
    st = synth.make_stack(cfg)
    pp = orc.make_psi_phi(st.sci, st.var, st.mask, st.psf)
    _, _, info = binding.debug_staged_plan(st.times, cfg.N, cfg.H, cfg.W, st.vel_grid, geom)
    assert info["CAP"] == {1: 6144, 2: 4096, 3: 6144}[geom]
    check_against_oracle(orc, pp, st.times, st.vel_grid, geom=geom)


def test_plan_interior_trajectories(orc):
    pp = synth.random_psiphi(9, 95, 200, seed=21, invalid_frac=0.03)
    times = np.array([0, .05, .1, .15, 1, 1.05, 1.1, 2.0, 2.05])
    vel = synth.velocity_grid(12, 10, -math.pi / 3, math.pi / 3, 3.0, 40.0)
    check_against_oracle(orc, pp, times, vel)


def test_plan_half_integer_and_near_tie_shifts(orc):
    """Velocities whose v*dt are exact halves or within an ulp of one at W = 4096: the pairs for
    which one integer shift is NOT the definition must come out as literal (unsafe) entries."""
    H, W = 33, 4096
    pp = np.zeros((3, H, W, 2), np.float32)
    pp[1:, ..., 0] = (np.arange(H)[:, None] * W + np.arange(W)[None, :]).astype(np.float32)[None]
    pp[..., 1] = 1.0
    times = np.array([0.0, 0.5, 1.0])
    vel = np.array([[3.0, 1.0], [-3.0, -1.0], [1.0, 3.0], [10.49999, 0.0], [20.99998, 0.5],
                    [0.49999997, 0.49999997], [0.99999994, -0.99999994], [7.0, 7.0],
                    [-0.5, 0.0], [2047.5, 0.0], [4095.0, 1.0], [10.5, 10.5]], np.float32)
    stream, _, info = binding.debug_staged_plan(times, 3, H, W, vel)
    assert ((stream[:, 0] & 0xFF) == ENT_UNSAFE).sum() >= 1
    tiles = [(0, 0), (31, 0), (63, 1), (40, 1)]
    check_against_oracle(orc, pp, times, vel, tiles)


def test_plan_degenerate_shapes(orc):
    # N = 1: no image to shift, one NOP|LAST entry per block
    pp = synth.random_psiphi(1, 1, 33, seed=1, invalid_frac=0.2)
    stream, _, info = binding.debug_staged_plan([3.0], 1, 1, 33, np.zeros((1, 2), np.float32))
    assert stream.shape[0] == 1 and (stream[0, 0] & 0xFF) == ENT_NOP and (stream[0, 0] >> 8) & FLAG_LAST
    check_against_oracle(orc, pp, [3.0], np.zeros((1, 2), np.float32))
    # velocities far beyond the image, unsorted times, duplicated velocities, V not a multiple of B
    pp = synth.random_psiphi(5, 37, 70, seed=3, invalid_frac=0.1)
    vel = synth.velocity_grid(4, 4, -2, 2, 2, 12)
    vel = np.concatenate([vel, vel[3:9], vel[:2], np.array([[5e4, 0], [0, -7e4], [3e3, 3e3]], np.float32)])
    times = np.array([5.0, 4.5, 6.0, 5.25, 7.0])
    check_against_oracle(orc, pp, times, vel)


def test_plan_maximum_image_count(orc):
    """N = 64 = KBMOD_MAX_IMAGES and N = 40 (the additive-count variants of the kernel)."""
    rng = np.random.default_rng(64)
    for N in (64, 40):
        pp = synth.random_psiphi(N, 40, 70, seed=N, invalid_frac=0.05)
        times = np.sort(rng.uniform(0.0, 5.0, N))
        vel = synth.velocity_grid(6, 4, -math.pi / 2, math.pi / 2, 1.0, 9.0)
        check_against_oracle(orc, pp, times, vel)


def test_fill_bytes_per_sample_byte_at_the_bench_workload():
    """The numbers of DESIGN.md section 5.2, recomputed: bytes the staged kernel's plan moves into shared
    memory per algorithmic sample byte at BASELINE.json configs[2] (15 x 4096 x 4096, 640 velocities),
    against the floor no grouping into boxes can beat -- the exact area of the union of a block's
    eight shifted 64 x 30 windows, rasterised here independently of the planner."""
    cfg = synth.config(3)
    times = synth.make_times(cfg, np.random.default_rng(cfg.seed))
    vel = synth.velocity_grid(cfg.n_angles, cfg.n_speeds, cfg.ang_lo, cfg.ang_hi, cfg.speed_lo, cfg.speed_hi)
    fills = {}
    for geom in (0, 1):
        stream, shapes, info = binding.debug_staged_plan(times, cfg.N, cfg.H, cfg.W, vel, geom)
        tma = stream[(stream[:, 0] & 0xFF) == 1]
        bw, bh = tma[:, 4] & 0xFFFF, tma[:, 4] >> 16
        assert (bw * bh <= info["CAP"]).all() and (bw % 2 == 0).all()
        fills[geom] = float((bw.astype(np.int64) * bh).sum()) / (cfg.V * cfg.N * info["TW"] * info["TH"])
        order = stream[(stream[:, 0] >> 8) & 1 == 1][:, 8 + info["B"]:8 + 2 * info["B"]]      # velocities of every block
    assert 0.66 < fills[1] < fills[0] < 0.72, fills            # 0.675 (cap 6144) and 0.692 (cap 4096)
    # exact union of the windows of every block and image (image 0 is read once per block: not staged)
    dt = (times - times[0]).astype(np.float32)
    sh = np.floor(vel[:, None, :].astype(np.float64) * dt[None, :, None] + 0.5).astype(np.int64)
    TW, TH = info["TW"], info["TH"]
    union = 0
    for blk in order:
        js = blk[blk >= 0]
        for i in range(1, cfg.N):
            s = sh[js, i]
            x0, y0 = s[:, 0].min(), s[:, 1].min()
            g = np.zeros((s[:, 1].max() - y0 + TH, s[:, 0].max() - x0 + TW), bool)
            for sx, sy in s:
                g[sy - y0:sy - y0 + TH, sx - x0:sx - x0 + TW] = True
            union += int(g.sum())
    floor = union / (cfg.V * cfg.N * TW * TH)
    assert 0.55 < floor < 0.59, floor                          # 0.570: no plan of 64 x 30 x 8 blocks stages less
    assert fills[1] / floor < 1.25
