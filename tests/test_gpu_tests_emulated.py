"""The `-m gpu` test files and the C-ABI layer, exercised on the CPU (`-m "not gpu"`).

With KBMOD_GPU_TESTS_EMULATED=1 the GPU test files take tests/emulated_binding.py in place of the
ctypes binding: the product's own binding.py (a private, patched copy) over
tests/hostlogic/libkbmod_emul.so, the WHOLE library -- api.cu and every kernel file -- compiled with
g++ against the SIMT emulator, on CPU tensors.  A child pytest runs a part of the GPU tests that way
on every CPU run, so that (1) the success paths of the ABI layer (workspace layout, plans, options,
kbmod_search_host's pipeline, the dispatch of every call) execute somewhere before a GPU sees them,
and (2) a GPU test that is wrong -- a bad expectation, a misuse of the API -- fails on this machine
and not on the first B200 that runs it.  (It has already paid for itself: it found that an empty band
of start rows was refused because zero-sized result planes have NULL data pointers, and two wrong
expectations in new GPU tests.)  The whole of the small-size GPU tests, all four search kernels
included, passes this way (`KBMOD_GPU_TESTS_EMULATED=1 KBMOD_TEST_STAGED=1 KBMOD_TEST_QUEUED=1 pytest
-m gpu tests -k "not full_size"`, a few minutes); the subset below keeps the CPU suite short.
Nothing here says anything about hardware.
"""
import os
import subprocess
import sys

import pytest

from paper_1901_02492_b200 import synth

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def test_gpu_test_files_pass_against_the_emulated_library():
    env = dict(os.environ, KBMOD_GPU_TESTS_EMULATED="1")
    cp = subprocess.run([sys.executable, "-m", "pytest", "-x", "-q", "-p", "no:cacheprovider", "-m", "gpu",
                         "tests/test_zx_gpu_next_rows.py", "tests/test_gpu_parity.py", "-k",
                         "next_rows or edge_cases or half_integer or eval_trajectories or maximum_image or "
                         "(row_bands and 0) or psi_phi or host_entry or split or errors"],
                        cwd=ROOT, env=env, capture_output=True, text=True, timeout=1200)
    assert cp.returncode == 0, cp.stdout[-4000:] + cp.stderr[-2000:]
    assert " passed" in cp.stdout and " failed" not in cp.stdout


def test_full_size_helper_on_a_small_stack(orc, monkeypatch):
    """The body shared by the full-size tests of every BASELINE.json config (psi/phi bands compared
    through a cropped oracle run with the PSF halo, search bands compared bit for bit), on a stack
    small enough for the emulator: image edges, a tile seam and the interior."""
    monkeypatch.setenv("KBMOD_GPU_TESTS_EMULATED", "1")
    import importlib
    from tests import emulated_binding, test_gpu_parity as P
    P = importlib.reload(P)
    try:
        cfg = synth.config(4, N=4, H=70, W=132, n_sources=3, n_angles=6, n_speeds=4, min_obs=3)
        res = P._full_size_case(emulated_binding, orc, cfg, (0, 28, 41, cfg.H - 8))
        assert res["nu"].shape == (cfg.H, cfg.W, cfg.K)
    finally:
        monkeypatch.delenv("KBMOD_GPU_TESTS_EMULATED")
        importlib.reload(P)
