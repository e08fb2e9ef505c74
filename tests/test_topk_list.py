"""S6 list code of the staged kernel (csrc/topk_list.h), compiled for the host: every insertion
sequence must leave the K best candidates in (nu descending, index ascending) order -- the
oracle's rule (Q15) -- for both the register variant (K <= 8) and the generic one."""
import ctypes
import os
import subprocess

import numpy as np
import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
SRC = os.path.join(ROOT, "tests", "hostlogic", "topk_host.cpp")
LIB = os.path.join(ROOT, "tests", "hostlogic", "libtopk_host.so")
EMPTY = 0x7FFFFFFF


@pytest.fixture(scope="module")
def topk():
    subprocess.run(["g++", "-O2", "-std=c++17", "-shared", "-fPIC", "-I",
                    os.path.join(ROOT, "paper_1901_02492_b200", "csrc"), SRC, "-o", LIB], check=True)
    L = ctypes.CDLL(LIB)
    L.host_list_insert.argtypes = [ctypes.c_int, ctypes.c_void_p, ctypes.c_void_p, ctypes.c_int,
                                   ctypes.c_float, ctypes.c_int]
    return L


def reference(cands, K):
    best = sorted(cands, key=lambda c: (-c[0], c[1]))[:K]
    nu = [c[0] for c in best] + [-np.inf] * (K - len(best))
    idx = [c[1] for c in best] + [EMPTY] * (K - len(best))
    return np.array(nu, np.float32), np.array(idx, np.int32)


@pytest.mark.parametrize("kp,K", [(8, 8), (8, 4), (8, 1), (8, 5), (0, 8), (0, 16), (0, 32), (0, 1), (0, 3)])
def test_insert_sequences(topk, kp, K):
    rng = np.random.default_rng(100 * kp + K)
    for trial in range(200):
        n = int(rng.integers(0, 60))
        # few distinct values => many exact ties; include -0.0/+0.0 and negative nu
        vals = rng.choice(np.array([-3.5, -0.0, 0.0, 1.25, 2.5, 7.0, 7.0000005], np.float32), n) \
            if trial % 2 else rng.standard_normal(n).astype(np.float32)
        idx = rng.permutation(1000)[:n]
        Ln = np.full(K, -np.inf, np.float32)
        Lj = np.full(K, EMPTY, np.int32)
        cands = []
        for v, j in zip(vals, idx):
            assert topk.host_list_insert(kp, Ln.ctypes.data, Lj.ctypes.data, K, float(v), int(j)) == 0
            cands.append((float(v), int(j)))
        rn, rj = reference(cands, K)
        assert (Lj == rj).all(), (trial, Lj, rj)
        assert (Ln == rn).all()


def test_order_independence(topk):
    """The final list does not depend on the order in which candidates arrive (the kernel
    visits velocities in Hilbert order and drains its queue in batches)."""
    rng = np.random.default_rng(5)
    vals = rng.integers(0, 6, 40).astype(np.float32)
    idx = np.arange(40)
    outs = []
    for _ in range(5):
        perm = rng.permutation(40)
        Ln = np.full(8, -np.inf, np.float32)
        Lj = np.full(8, EMPTY, np.int32)
        for p in perm:
            topk.host_list_insert(8, Ln.ctypes.data, Lj.ctypes.data, 8, float(vals[p]), int(idx[p]))
        outs.append((Ln.copy(), Lj.copy()))
    for a, b in outs[1:]:
        assert (a == outs[0][0]).all() and (b == outs[0][1]).all()
