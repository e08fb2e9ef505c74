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


HARNESSES = {"tiled_simt": "1", "staged_simt": '"simt_ptx.h"', "post_simt": "1"}


def build_command(name, sanitize=SANITIZE):
    """(library path, g++ command) of tests/hostlogic/<name>.cpp (which includes csrc/*.cu files)."""
    src = os.path.join(HL, name + ".cpp")
    lib = os.path.join(HL, f"lib{name}{'_asan' if sanitize else ''}.so")
    cmd = ["g++", "-O1", "-std=c++17", "-ffp-contract=off", "-shared", "-fPIC",
           "-I", os.path.join(HL, "simt"), "-I", os.path.join(ROOT, "include"), "-I", CSRC,
           f"-DKBMOD_SIMT_EMUL={HARNESSES[name]}", *(SAN_FLAGS if sanitize else []), src, "-o", lib]
    return lib, cmd


_running = {}        # library path -> Popen of the g++ that is building it (this process started it)


def _start(name, sanitize):
    lib, cmd = build_command(name, sanitize)
    if lib not in _running and _stale(lib, os.path.join(HL, name + ".cpp")):
        _running[lib] = subprocess.Popen(cmd)
    return lib


def _wait(lib, what):
    p = _running.pop(lib, None)
    if p is not None and p.wait() != 0:
        raise RuntimeError(f"g++ failed on {what}")


def start_background_builds(sanitized=True):
    """Starts every stale harness build at once and returns immediately (tests/conftest.py calls this
    at session start, so the compilers run while the first tests do); load() / build_all() wait for
    the library they need."""
    for name in HARNESSES:
        _start(name, False)
        if sanitized:
            _start(name, True)


def build_all(sanitize=SANITIZE):
    """Compiles every stale harness of one flavour, all at once (they are independent translation units)."""
    libs = [(name, _start(name, sanitize)) for name in HARNESSES]
    for name, lib in libs:
        _wait(lib, name)


def load(name, emul_define=None):
    """Compiles tests/hostlogic/<name>.cpp if stale and loads it."""
    lib = _start(name, SANITIZE)
    _wait(lib, name)
    return ctypes.CDLL(lib)


# ---- the whole C-ABI library under emulation (tests/hostlogic/abi_simt.cpp)
ABI_SOURCES = ["api.cu", "psi_phi.cu", "search_direct.cu", "search_tiled.cu", "search_staged.cu", "postproc.cu"]


def build_abi_lib():
    """Compiles every csrc/*.cu (one translation unit each, in parallel) plus the glue with g++ against
    the SIMT emulator and links tests/hostlogic/libkbmod_emul.so; returns its path."""
    lib = os.path.join(HL, "libkbmod_emul.so")
    glue = os.path.join(HL, "abi_simt.cpp")
    if not _stale(lib, glue):
        return lib
    out = os.path.join(HL, "build_abi")
    os.makedirs(out, exist_ok=True)
    flags = ["-O1", "-std=c++17", "-ffp-contract=off", "-fPIC", "-fno-gnu-unique", "-I", os.path.join(HL, "simt"),
             "-I", os.path.join(ROOT, "include"), "-I", CSRC, '-DKBMOD_SIMT_EMUL="simt_ptx.h"']
    procs, objs = [], []
    for src in [os.path.join(CSRC, f) for f in ABI_SOURCES] + [glue]:
        obj = os.path.join(out, os.path.basename(src) + ".o")
        objs.append(obj)
        procs.append((src, subprocess.Popen(["g++", *flags, "-x", "c++", "-c", src, "-o", obj])))
    for src, p in procs:
        if p.wait() != 0:
            raise RuntimeError(f"g++ failed on {src}")
    # -Bsymbolic: the library binds its own symbols (the emulator state, smem_raw) whatever else is loaded
    subprocess.run(["g++", "-shared", "-Wl,-Bsymbolic", "-o", lib, *objs], check=True)
    return lib
