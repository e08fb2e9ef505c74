"""The staged kernel's shared-memory ring allocator (csrc/ring_alloc.h), compiled for the host:
FIFO allocations of random sizes with a lagging consumer must never overlap, must stay inside the
ring and 128-byte aligned (TMA destination), and must always make progress."""
import ctypes
import os
import subprocess

import numpy as np
import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
SRC = os.path.join(ROOT, "tests", "hostlogic", "ring_host.cpp")
LIB = os.path.join(ROOT, "tests", "hostlogic", "libring_host.so")


@pytest.fixture(scope="module")
def ring():
    subprocess.run(["g++", "-O2", "-std=c++17", "-shared", "-fPIC", "-I",
                    os.path.join(ROOT, "paper_1901_02492_b200", "csrc"), SRC, "-o", LIB], check=True)
    return ctypes.CDLL(LIB)


def run(ring, which, sizes, lag):
    sizes = np.ascontiguousarray(sizes, np.uint32)
    lag = np.ascontiguousarray(lag, np.uint32)
    offs = np.zeros(len(sizes), np.uint32)
    peak = ctypes.c_longlong(0)
    rc = ring.host_ring_simulate(which, sizes.ctypes.data_as(ctypes.c_void_p), len(sizes),
                                 lag.ctypes.data_as(ctypes.c_void_p), offs.ctypes.data_as(ctypes.c_void_p),
                                 ctypes.byref(peak))
    return rc, offs, peak.value


@pytest.mark.parametrize("seed", range(6))
def test_random_streams_big_ring(ring, seed):
    rng = np.random.default_rng(seed)
    n = 20000
    # box sizes as the plan produces them (15-48 KB), empty entries (NOP / unsafe / off-image), rare full-cap boxes
    sizes = (rng.integers(120, 385, n) * 128).astype(np.uint32)
    sizes[rng.random(n) < 0.15] = 0
    sizes[rng.random(n) < 0.01] = 49152
    lag = rng.integers(0, 20, n)
    rc, offs, peak = run(ring, 0, sizes, lag)
    assert rc == 0
    assert peak > 150000          # the ring really is used deeply (> 150 KB live at some point)


@pytest.mark.parametrize("seed", range(4))
def test_tiny_ring_edge_cases(ring, seed):
    """4 KB ring, 4 header slots: exact fits, wraps with skipped tails, entries as big as the ring."""
    rng = np.random.default_rng(100 + seed)
    n = 5000
    sizes = (rng.integers(0, 33, n) * 128).astype(np.uint32)          # 0 .. 4096
    lag = rng.integers(0, 6, n)
    rc, offs, peak = run(ring, 1, sizes, lag)
    assert rc == 0 and peak <= 4096
    # deterministic corner: ring-sized entries back to back, and all-empty streams
    assert run(ring, 1, [4096] * 10, [5] * 10)[0] == 0
    assert run(ring, 1, [0] * 50, [3] * 50)[0] == 0
    assert run(ring, 1, [2048, 2048, 2048, 1024, 3072, 128, 4096], [9] * 7)[0] == 0
