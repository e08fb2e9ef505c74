// tests/hostlogic/abi_simt.cpp -- TEST INFRASTRUCTURE.  The glue of the EMULATED C-ABI library
// (tests/hostlogic/libkbmod_emul.so): every csrc/*.cu file of the product -- api.cu included --
// compiled with g++ against the SIMT emulator as its own translation unit and linked together, so
// that the whole library behind include/kbmod_b200.h (argument checks, workspace layout, host plans,
// launch code, kernels) runs on host memory.  tests/emulated_binding.py loads it in place of
// libkbmod_b200.so to exercise the ABI layer and the -m gpu test files' logic without a GPU.  This
// file only owns the emulated CTA's shared-memory array.  Not part of the product.
#include <cuda.h>
#include <cuda_runtime.h>

namespace kbmod {
alignas(1024) unsigned char smem_raw[simt::SMEM_MAX + 64];
}  // namespace kbmod

namespace {
struct Init {
    Init() { simt::S().smem = kbmod::smem_raw; }
} init_shared_memory;
}  // namespace
