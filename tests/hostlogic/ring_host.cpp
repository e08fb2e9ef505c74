// Host build of csrc/ring_alloc.h for tests/test_ring_alloc.py: a producer that allocates `n`
// entries of the given sizes while a consumer releases them in order with a random lag.
// Returns 0 if no two live entries ever overlapped and every entry was placed, else a code.
#include <cstdint>
#include <vector>

#include "ring_alloc.h"

template <int RB, int NH>
static int simulate(const uint32_t* bytes, int n, const uint32_t* lag, uint32_t* offs, long long* max_live_bytes) {
    unsigned adv[NH];
    kbmod::RingAlloc<RB, NH> ring(adv);
    struct Live { long long g; unsigned off, len; };
    std::vector<Live> live;
    long long peak = 0;
    for (int g = 0; g < n; ++g) {
        if (bytes[g] % 128 || bytes[g] > (uint32_t)RB) return 1;
        // the consumer has finished everything older than g - lag[g]
        int spins = 0;
        for (;;) {
            while (!live.empty() && live.front().g < (long long)g - (long long)lag[g] && ring.in_flight()) {
                if (live.front().g != ring.oldest) return 2;          // FIFO order broken
                ring.release_oldest();
                live.erase(live.begin());
            }
            if (ring.fits(bytes[g])) break;
            // the producer would now wait for entry `oldest`: it must exist, else deadlock
            if (!ring.in_flight()) return 3;
            if (live.front().g != ring.oldest) return 2;
            ring.release_oldest();
            live.erase(live.begin());
            if (++spins > 4 * NH) return 4;
        }
        const unsigned off = ring.place(bytes[g]);
        if (off % 128 || off + bytes[g] > (unsigned)RB) return 5;
        for (const Live& l : live)
            if (l.len && bytes[g] && off < l.off + l.len && l.off < off + bytes[g]) return 6;   // overlap
        live.push_back({g, off, bytes[g]});
        if ((int)live.size() > NH) return 7;
        long long sum = 0;
        for (const Live& l : live) sum += l.len;
        if (sum > peak) peak = sum;
        offs[g] = off;
    }
    *max_live_bytes = peak;
    return 0;
}

extern "C" int host_ring_simulate(int which, const uint32_t* bytes, int n, const uint32_t* lag, uint32_t* offs,
                                  long long* max_live_bytes) {
    if (which == 0) return simulate<212992, 16>(bytes, n, lag, offs, max_live_bytes);
    if (which == 1) return simulate<4096, 4>(bytes, n, lag, offs, max_live_bytes);
    return -1;
}
