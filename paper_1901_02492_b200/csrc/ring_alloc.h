// ring_alloc.h -- byte-granular FIFO allocator for the staged kernel's shared-memory data ring.
//
// The producer warp of search_staged_kernel stages TMA boxes of different sizes; consumers
// release them strictly in order.  Live data is therefore one contiguous run (in ring order)
// that ends at `head`; `used` is its length including the bytes skipped when an allocation did
// not fit before the end of the ring.  Entry g records in adv[g % NH] how far it advanced
// `head`, so that releasing the oldest entry just subtracts that amount.  Plain integers, no
// memory accesses besides the small adv[] table: the same code runs on the device and in the
// host unit test (tests/test_ring_alloc.py).
#pragma once

#if defined(__CUDACC__)
#define KBMOD_RA_HD __host__ __device__ __forceinline__
#else
#define KBMOD_RA_HD inline
#endif

namespace kbmod {

template <int RING_BYTES, int NH>
struct RingAlloc {
    unsigned head = 0;          // next allocation offset
    unsigned used = 0;          // bytes between the oldest live entry's start and head (ring order)
    long long oldest = 0;       // index of the oldest entry not yet released
    long long next = 0;         // index of the next entry to allocate
    unsigned* adv;              // [NH] bytes each in-flight entry advanced head by

    KBMOD_RA_HD explicit RingAlloc(unsigned* adv_table) : adv(adv_table) {}

    // true if entry `next` may be placed now: its header slot (next % NH) is free and `bytes`
    // (a multiple of 128, <= RING_BYTES) fit.  Otherwise the caller must release_oldest() (after
    // waiting for the consumers of entry `oldest`) and ask again.
    KBMOD_RA_HD bool fits(unsigned bytes) const {
        if (next - oldest >= NH) return false;                    // header slot still in use
        if (used == 0) return true;                               // empty ring: restart at 0
        if (head + bytes <= (unsigned)RING_BYTES) return used + bytes <= (unsigned)RING_BYTES;
        return used + ((unsigned)RING_BYTES - head) + bytes <= (unsigned)RING_BYTES;   // wrap
    }

    // places entry `next` (fits(bytes) must hold) and returns its data offset
    KBMOD_RA_HD unsigned place(unsigned bytes) {
        if (used == 0) head = 0;
        unsigned off = head, step = bytes;
        if (head + bytes > (unsigned)RING_BYTES) {                // skip the tail of the ring
            step += (unsigned)RING_BYTES - head;
            off = 0;
        }
        head = off + bytes;
        if (head == (unsigned)RING_BYTES) head = 0;
        used += step;
        adv[next % NH] = step;
        ++next;
        return off;
    }

    KBMOD_RA_HD bool in_flight() const { return oldest < next; }

    // the consumers are done with entry `oldest`
    KBMOD_RA_HD void release_oldest() {
        used -= adv[oldest % NH];
        ++oldest;
    }
};

}  // namespace kbmod
