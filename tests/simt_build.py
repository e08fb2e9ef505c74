"""Builds the SIMT-emulation harnesses of tests/hostlogic/ (TEST INFRASTRUCTURE).

Two flavours of every harness:
  plain      g++ -O1                                   -> lib<name>.so        (loaded by the pytest process)
  sanitized  g++ -O1 -g -fsanitize=address,undefined   -> lib<name>_asan.so   (KBMOD_SIMT_SANITIZE=1)
The sanitized flavour needs the ASan runtime first in the process's library list, so it is only
loaded by a child interpreter started with LD_PRELOAD=libasan (tests/test_simt_sanitized.py).
"""
import ctypes
import os
import subprocess

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
HL = os.path.join(ROOT, "tests", "hostlogic")
CSRC = os.path.join(ROOT, "paper_1901_02492_b200", "csrc")
SANITIZE = os.environ.get("KBMOD_SIMT_SANITIZE") == "1"
SAN_FLAGS = ["-g", "-fno-omit-frame-pointer", "-fsanitize=address,undefined", "-fno-sanitize-recover=all"]


def _stale(lib, src):
    if not os.path.exists(lib):
        return True
    t = os.path.getmtime(lib)
    deps = [src, os.path.join(ROOT, "include", "kbmod_b200.h")]
    deps += [os.path.join(CSRC, f) for f in os.listdir(CSRC)]
    deps += [os.path.join(HL, "simt", f) for f in os.listdir(os.path.join(HL, "simt"))]
    return any(os.path.getmtime(d) > t for d in deps)


def load(name, emul_define):
    """Compiles tests/hostlogic/<name>.cpp (which includes a csrc/*.cu file) if stale and loads it."""
    src = os.path.join(HL, name + ".cpp")
    lib = os.path.join(HL, f"lib{name}{'_asan' if SANITIZE else ''}.so")
    if _stale(lib, src):
        cmd = ["g++", "-O1", "-std=c++17", "-ffp-contract=off", "-shared", "-fPIC",
               "-I", os.path.join(HL, "simt"), "-I", os.path.join(ROOT, "include"), "-I", CSRC,
               f"-DKBMOD_SIMT_EMUL={emul_define}", *(SAN_FLAGS if SANITIZE else []), src, "-o", lib]
        subprocess.run(cmd, check=True)
    return ctypes.CDLL(lib)
