"""The SIMT-emulation tests again, under AddressSanitizer + UBSan (`-m "not gpu"`).

An out-of-bounds global load or store is an illegal address on the GPU (Xid 13/31).  The plain
emulation build would read or corrupt a neighbouring host allocation silently, so a seeded subset
of tests/test_tiled_simt.py and tests/test_staged_simt.py and the whole of tests/test_post_simt.py
are re-run here in child interpreters with the harnesses compiled with -fsanitize=address,undefined
(tests/simt_build.py) and every emulated device buffer a heap block of exactly the size the product
gives the kernel (hostlogic/simt/devmem.h; the shared-memory array is poisoned beyond the launch's
dynamic size).  Any such access aborts the child and fails the test.  The oracle is built the same
way and re-runs its pins (S:section 5 "sanitizers").  The children run concurrently.
"""
import os
import subprocess
import sys

import pytest

from tests import simt_build

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
pytestmark = pytest.mark.skipif(os.environ.get("KBMOD_SIMT_SANITIZE") == "1",
                                reason="already inside the sanitized child")

CHILDREN = {
    # kernels 2 and 4 (search_tiled.cu): config 1, the K = 16 crop, degenerate shapes, image counts, the
    # limit cases, row bands and the seeded randomized problems
    "tiled": ["tests/test_tiled_simt.py", "-k",
              "config1 or (crops and over2) or degenerate or image_count or limit or band or randomized"],
    # kernel 3 (search_staged.cu): config 1 under all schedules, the K = 16 crop, limit cases, row bands,
    # every ring geometry, literal-shift entries, image counts, randomized problems on ring 0
    "staged": ["tests/test_staged_simt.py", "-k",
               "config1 or (crops and over2) or limit or band or geometr or degenerate or unproven or image_count "
               "or (randomized and 0)"],
    # search_direct.cu (top-K, threshold), postproc.cu (N1 filter, N2 stamps, N3 mask builder) and the
    # threshold mode of the queued tiled kernel
    "post": ["tests/test_post_simt.py"],
    # oracle.c itself on all its pins
    "oracle": ["tests/test_oracle_pins.py", "tests/test_oracle_next_rows.py"],
}


def _asan_runtime():
    p = subprocess.run(["gcc", "-print-file-name=libasan.so"], capture_output=True, text=True).stdout.strip()
    return p if os.path.isabs(p) and os.path.exists(p) else None


def _env(rt):
    return dict(os.environ, LD_PRELOAD=rt, KBMOD_SIMT_SANITIZE="1", KBMOD_ORACLE_SANITIZE="1",
                ASAN_OPTIONS="detect_leaks=0:abort_on_error=1:halt_on_error=1",
                UBSAN_OPTIONS="print_stacktrace=1:halt_on_error=1")


@pytest.fixture(scope="module")
def children(tmp_path_factory):
    rt = _asan_runtime()
    if rt is None:
        pytest.skip("gcc has no libasan.so on this machine")
    simt_build.build_all(sanitize=True)                 # the three harnesses, compiled side by side
    # the sanitized oracle is built ONCE here: every child loads it, none may find it half written
    subprocess.run([sys.executable, "-c", "import oracle; oracle.build()"], cwd=ROOT, check=True,
                   env=dict(os.environ, KBMOD_ORACLE_SANITIZE="1"))
    d = tmp_path_factory.mktemp("sanitized")
    procs = {}
    for name, args in CHILDREN.items():
        out = open(d / f"{name}.log", "w")
        procs[name] = (subprocess.Popen([sys.executable, "-m", "pytest", "-x", "-q", "-p", "no:cacheprovider", *args],
                                        cwd=ROOT, env=_env(rt), stdout=out, stderr=subprocess.STDOUT), d / f"{name}.log")
    yield procs
    for p, _ in procs.values():
        if p.poll() is None:
            p.kill()


@pytest.mark.parametrize("name", list(CHILDREN))
def test_under_asan_ubsan(children, name):
    p, log = children[name]
    rc = p.wait(timeout=1500)
    text = open(log).read()
    assert rc == 0, f"sanitized child '{name}' failed (rc {rc}):\n{text[-4000:]}"
    assert " passed" in text and " failed" not in text, text[-2000:]


def test_the_detector_detects():
    """One element past an emulated device buffer through __ldg aborts the sanitized child with a
    heap-buffer-overflow report; the last element inside does not."""
    rt = _asan_runtime()
    if rt is None:
        pytest.skip("gcc has no libasan.so on this machine")
    env = dict(os.environ, LD_PRELOAD=rt, KBMOD_SIMT_SANITIZE="1", ASAN_OPTIONS="detect_leaks=0")
    code = ("import ctypes, sys; from tests import simt_build; L = simt_build.load('tiled_simt'); "
            "L.simt_selftest_ldg_past_end.restype = ctypes.c_ulonglong; "
            "L.simt_selftest_ldg_past_end(int(sys.argv[1])); print('survived')")
    ok = subprocess.run([sys.executable, "-c", code, "0"], cwd=ROOT, env=env, capture_output=True, text=True)
    assert ok.returncode == 0 and "survived" in ok.stdout, ok.stderr[-2000:]
    bad = subprocess.run([sys.executable, "-c", code, "1"], cwd=ROOT, env=env, capture_output=True, text=True)
    assert bad.returncode != 0 and "survived" not in bad.stdout
    assert "heap-buffer-overflow" in bad.stderr


def test_the_detector_detects_misaligned_vector_loads():
    """A 16-byte vector load 4 or 8 bytes off its alignment (a "misaligned address" fault on the GPU)
    aborts the sanitized child with UBSan's misaligned-address report; an aligned one does not."""
    rt = _asan_runtime()
    if rt is None:
        pytest.skip("gcc has no libasan.so on this machine")
    env = dict(os.environ, LD_PRELOAD=rt, KBMOD_SIMT_SANITIZE="1", ASAN_OPTIONS="detect_leaks=0",
               UBSAN_OPTIONS="print_stacktrace=1:halt_on_error=1")
    code = ("import ctypes, sys; from tests import simt_build; L = simt_build.load('tiled_simt'); "
            "L.simt_selftest_ldg128_misaligned.restype = ctypes.c_float; "
            "L.simt_selftest_ldg128_misaligned(int(sys.argv[1])); print('survived')")
    ok = subprocess.run([sys.executable, "-c", code, "0"], cwd=ROOT, env=env, capture_output=True, text=True)
    assert ok.returncode == 0 and "survived" in ok.stdout, ok.stderr[-2000:]
    for off in ("4", "8"):
        bad = subprocess.run([sys.executable, "-c", code, off], cwd=ROOT, env=env, capture_output=True, text=True)
        assert bad.returncode != 0 and "survived" not in bad.stdout, off
        assert "misaligned address" in bad.stderr, bad.stderr[-1500:]
