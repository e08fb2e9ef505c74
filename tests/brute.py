"""Independent brute force of the trajectory search for TINY stacks (pin P4).

Shares nothing with oracle/ or the CUDA path.  Pure Python loops.  Trajectory positions are
computed in exact rational arithmetic (fractions.Fraction) from the binary32 values of v
and dt; the caller must use cases where no position is within 1e-3 px of a pixel boundary,
so that the binary32 roundings of the definition cannot change the nearest pixel (this
function asserts it).  Sums in Python floats (binary64), selection by a full sort.  Beside the
binary64 sums the search also returns `psi32` / `phi32` / `nu32` / `alpha32`: the same samples
added in image order as numpy.float32 scalars (one IEEE binary32 rounding per add, divide and
sqrt), the bit-level definition of the oracle's f32seq mode (Q18).

Follows PAPER.md:193-197 Eq.24-26 and P:205 Eq.27 directly.
"""
from fractions import Fraction
import math

import numpy as np


def nearest_pixel(p0: int, v: np.float32, dt: np.float32) -> int:
    pos = Fraction(int(p0)) + Fraction(float(v)) * Fraction(float(dt)) + Fraction(1, 2)
    fl = math.floor(pos)
    frac = pos - fl
    assert Fraction(1, 1000) < frac < Fraction(999, 1000), "case too close to a pixel boundary"
    return fl


def search(psiphi: np.ndarray, times: np.ndarray, vel: np.ndarray, K: int, min_obs: int):
    N, H, W, _ = psiphi.shape
    V = vel.shape[0]
    dt = [np.float32(times[i] - times[0]) for i in range(N)]
    out = {k: np.zeros((H, W, K), np.float64) for k in ("psi", "phi", "nu", "alpha")}
    out["vel_idx"] = np.full((H, W, K), -1, np.int64)
    out["n_obs"] = np.zeros((H, W, K), np.int64)
    out["nu"][:] = -np.inf
    for k in ("psi32", "phi32", "nu32", "alpha32"):
        out[k] = np.zeros((H, W, K), np.float32)
    out["nu32"][:] = -np.inf
    for y0 in range(H):
        for x0 in range(W):
            cands = []
            for j in range(V):
                Psi = 0.0
                Phi = 0.0
                Psi32 = np.float32(0.0)
                Phi32 = np.float32(0.0)
                n = 0
                for i in range(N):
                    ix = nearest_pixel(x0, vel[j, 0], dt[i])
                    iy = nearest_pixel(y0, vel[j, 1], dt[i])
                    if not (0 <= ix < W and 0 <= iy < H):
                        continue
                    psi = float(psiphi[i, iy, ix, 0])
                    if math.isnan(psi):
                        continue
                    Psi += psi
                    Phi += float(psiphi[i, iy, ix, 1])
                    Psi32 = np.float32(Psi32 + psiphi[i, iy, ix, 0])      # binary32 add, image order
                    Phi32 = np.float32(Phi32 + psiphi[i, iy, ix, 1])
                    n += 1
                if n >= min_obs and Phi > 0:
                    cands.append((-Psi / math.sqrt(Phi), j, Psi, Phi, n, Psi32, Phi32))
            cands.sort()
            for k, (mnu, j, Psi, Phi, n, Psi32, Phi32) in enumerate(cands[:K]):
                out["psi32"][y0, x0, k] = Psi32
                out["phi32"][y0, x0, k] = Phi32
                out["nu32"][y0, x0, k] = np.float32(Psi32 / np.sqrt(Phi32))
                out["alpha32"][y0, x0, k] = np.float32(Psi32 / Phi32)
                out["vel_idx"][y0, x0, k] = j
                out["n_obs"][y0, x0, k] = n
                out["psi"][y0, x0, k] = Psi
                out["phi"][y0, x0, k] = Phi
                out["nu"][y0, x0, k] = -mnu
                out["alpha"][y0, x0, k] = Psi / Phi
    return out
