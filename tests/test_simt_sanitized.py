"""The SIMT-emulation tests again, under AddressSanitizer + UBSan (`-m "not gpu"`).

An out-of-bounds global load or store is an illegal address on the GPU (Xid 13/31).  The plain
emulation build would read or corrupt a neighbouring host allocation silently, so a seeded subset
of tests/test_tiled_simt.py and tests/test_staged_simt.py is re-run here in a child interpreter with
the harnesses compiled with -fsanitize=address,undefined (tests/simt_build.py) and every emulated
device buffer a heap block of exactly the size the product gives the kernel (hostlogic/simt/devmem.h;
the shared-memory array is poisoned beyond the launch's dynamic size).  Any such access aborts the
child and fails the test.  The oracle is built the same way once (S:section 5 "sanitizers").
"""
import os
import subprocess
import sys

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _asan_runtime():
    p = subprocess.run(["gcc", "-print-file-name=libasan.so"], capture_output=True, text=True).stdout.strip()
    return p if os.path.isabs(p) and os.path.exists(p) else None


def _run_child(args, timeout=1500):
    rt = _asan_runtime()
    if rt is None:
        pytest.skip("gcc has no libasan.so on this machine")
    env = dict(os.environ, LD_PRELOAD=rt, KBMOD_SIMT_SANITIZE="1", KBMOD_ORACLE_SANITIZE="1",
               ASAN_OPTIONS="detect_leaks=0:abort_on_error=1:halt_on_error=1",
               UBSAN_OPTIONS="print_stacktrace=1:halt_on_error=1")
    cp = subprocess.run([sys.executable, "-m", "pytest", "-x", "-q", "-p", "no:cacheprovider", *args],
                        cwd=ROOT, env=env, capture_output=True, text=True, timeout=timeout)
    tail = (cp.stdout[-3000:] + "\n" + cp.stderr[-3000:])
    assert cp.returncode == 0, f"sanitized child failed (rc {cp.returncode}):\n{tail}"
    assert " passed" in cp.stdout and "failed" not in cp.stdout, tail


@pytest.mark.skipif(os.environ.get("KBMOD_SIMT_SANITIZE") == "1", reason="already inside the sanitized child")
def test_the_detector_detects():
    """One element past an emulated device buffer through __ldg aborts the sanitized child with a
    heap-buffer-overflow report; the last element inside does not."""
    rt = _asan_runtime()
    if rt is None:
        pytest.skip("gcc has no libasan.so on this machine")
    env = dict(os.environ, LD_PRELOAD=rt, KBMOD_SIMT_SANITIZE="1", ASAN_OPTIONS="detect_leaks=0")
    code = ("import ctypes, sys; from tests import simt_build; L = simt_build.load('tiled_simt', '1'); "
            "L.simt_selftest_ldg_past_end.restype = ctypes.c_ulonglong; "
            "L.simt_selftest_ldg_past_end(int(sys.argv[1])); print('survived')")
    ok = subprocess.run([sys.executable, "-c", code, "0"], cwd=ROOT, env=env, capture_output=True, text=True)
    assert ok.returncode == 0 and "survived" in ok.stdout, ok.stderr[-2000:]
    bad = subprocess.run([sys.executable, "-c", code, "1"], cwd=ROOT, env=env, capture_output=True, text=True)
    assert bad.returncode != 0 and "survived" not in bad.stdout
    assert "heap-buffer-overflow" in bad.stderr


@pytest.mark.skipif(os.environ.get("KBMOD_SIMT_SANITIZE") == "1", reason="already inside the sanitized child")
def test_tiled_kernels_under_asan_ubsan():
    """Kernels 2 and 4 (search_tiled.cu): config 1, the K = 16 crop, degenerate shapes, image counts,
    the limit cases, row bands and the seeded randomized problems (about half a minute of emulation)."""
    _run_child(["tests/test_tiled_simt.py", "-k",
                "config1 or (crops and over2) or degenerate or image_count or limit or band or randomized"])


@pytest.mark.skipif(os.environ.get("KBMOD_SIMT_SANITIZE") == "1", reason="already inside the sanitized child")
def test_staged_kernel_under_asan_ubsan():
    """Kernel 3 (search_staged.cu): config 1 under all schedules, the K = 16 crop, limit cases, row
    bands, every ring geometry, literal-shift entries, image counts, randomized problems on ring 0."""
    _run_child(["tests/test_staged_simt.py", "-k",
                "config1 or (crops and over2) or limit or band or geometr or degenerate or unproven or image_count "
                "or (randomized and 0)"])


@pytest.mark.skipif(os.environ.get("KBMOD_SIMT_SANITIZE") == "1", reason="already inside the sanitized child")
def test_oracle_under_asan_ubsan():
    """oracle.c itself with -fsanitize=address,undefined on the pins that exercise every function."""
    _run_child(["tests/test_oracle_pins.py"])
