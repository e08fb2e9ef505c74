// tests/hostlogic/simt/devmem.h -- TEST INFRASTRUCTURE: emulated "device" allocations of EXACT size.
//
// The SIMT-emulation harnesses hand the kernels host memory in place of device memory.  Every such
// buffer is its own heap block of exactly the number of bytes the product would give the kernel, so
// that under -fsanitize=address an out-of-bounds __ldg / __stcg / TMA source read -- an illegal
// address on the GPU (Xid 13/31) -- lands in a redzone and aborts the test instead of reading or
// corrupting a neighbour silently (tests/test_simt_sanitized.py runs the harnesses that way).
#pragma once
#include <stdlib.h>
#include <string.h>

namespace simt {

struct DevBuf {
    void* p = nullptr;
    size_t n = 0;
    explicit DevBuf(size_t bytes, size_t align = 256, int fill = 0xA5) : n(bytes) {
        // posix_memalign: exact user size (no rounding to the alignment), so the right redzone
        // starts at byte n; a zero-sized buffer still gets a distinct address
        if (posix_memalign(&p, align, bytes ? bytes : 1) != 0) abort();
        memset(p, fill, bytes);
    }
    DevBuf(const void* src, size_t bytes, size_t align = 256) : DevBuf(bytes, align) { memcpy(p, src, bytes); }
    ~DevBuf() { free(p); }
    DevBuf(const DevBuf&) = delete;
    DevBuf& operator=(const DevBuf&) = delete;
    template <class T> T* as() { return static_cast<T*>(p); }
    void copy_to(void* dst) const { memcpy(dst, p, n); }
};

}  // namespace simt
