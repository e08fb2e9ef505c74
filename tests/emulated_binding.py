"""TEST INFRASTRUCTURE: the product's own binding (paper_1901_02492_b200/binding.py, loaded a second
time under another module name) over the EMULATED C-ABI library tests/hostlogic/libkbmod_emul.so --
every csrc/*.cu file of the product, api.cu included, compiled with g++ against the SIMT emulator
(tests/simt_build.build_abi_lib) -- on CPU tensors.

It exists so that, on a machine without a GPU, (1) the success paths of the ABI layer run at all:
argument marshalling, workspace layout, host plans, kbmod_search_host's copy / build / search /
copy-back sequence, the dispatch of every kernel and option; and (2) the LOGIC of the `-m gpu` test
files -- their cases, expectations and use of the API -- is exercised
(`KBMOD_GPU_TESTS_EMULATED=1 pytest -m gpu ...`; tests/test_gpu_tests_emulated.py runs a part of
that in the CPU suite).  It proves nothing about hardware.  The product file is not modified and has
no such mode: this module patches its own private copy (library path, "is a CUDA tensor" check,
stream handle).  Not part of the product; the product has no CPU path.
"""
import ctypes
import importlib.util
import os
import sys

import torch as _torch

from tests import simt_build

_ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
_spec = importlib.util.spec_from_file_location("kbmod_binding_emulated",
                                               os.path.join(_ROOT, "paper_1901_02492_b200", "binding.py"))
_b = importlib.util.module_from_spec(_spec)
sys.modules["kbmod_binding_emulated"] = _b
_spec.loader.exec_module(_b)
_b.LIB_PATH = simt_build.build_abi_lib()


def _dev(t, dtype, what):
    """As binding._dev, for the emulated library's "device" = host memory."""
    if t is None:
        return None
    if not (isinstance(t, _torch.Tensor) and not t.is_cuda and t.dtype == dtype and t.is_contiguous()):
        raise _b.KbmodError(f"{what}: expected a contiguous tensor of {dtype}")
    return ctypes.c_void_p(t.data_ptr())


_b._dev = _dev
_b._stream = lambda: ctypes.c_void_p(0)


def aligned_empty(n, align=256):
    """A uint8 CPU tensor of n bytes whose data pointer is `align`-byte aligned (CUDA allocations are
    512-byte aligned; the CPU allocator only guarantees 64, the ABI asks 256 for workspaces)."""
    raw = _torch.empty(int(n) + align, dtype=_torch.uint8)
    off = (-raw.data_ptr()) % align
    return raw[off:off + int(n)]


_b.alloc_workspace = lambda nbytes, device=None: aligned_empty(nbytes)

# the public names of the binding, served by the patched copy
for _name in dir(_b):
    if not _name.startswith("_") and _name not in ("torch", "np", "ctypes", "os", "annotations"):
        globals()[_name] = getattr(_b, _name)


def set_search_kernel(which):
    _b.set_search_kernel(which)
