import os
import sys

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)


def pytest_configure(config):
    config.addinivalue_line("markers", "gpu: needs a CUDA device (run on the B200 box)")


def pytest_sessionstart(session):
    """CPU runs: start compiling the SIMT-emulation harnesses (plain and sanitized) right away, in the
    background, so that the compilers work while the first tests run (tests/simt_build.py)."""
    if session.config.getoption("markexpr", "") == "gpu" or os.environ.get("KBMOD_SIMT_SANITIZE") == "1" \
            or os.environ.get("KBMOD_GPU_TESTS_EMULATED") == "1":
        return
    try:
        from tests import simt_build
        simt_build.start_background_builds()
    except Exception:
        pass                     # a fixture will report the build failure where it matters


@pytest.fixture(scope="session")
def orc():
    """The CPU oracle (tests may use it; the product never does)."""
    import oracle
    oracle.build()
    return oracle
