// search_common.cuh -- pieces shared by the tiled (search_tiled.cu) and staged (search_staged.cu)
// search kernels: the velocity processing order and the S5 pre-test / queue step.
#pragma once
#include <algorithm>
#include <utility>
#include <vector>

#include "common.cuh"

namespace kbmod {

// Hilbert index of a 16-bit quantised (x, y)
inline unsigned hilbert_d(unsigned x, unsigned y) {
    unsigned d = 0;
    for (unsigned s = 1u << 15; s > 0; s >>= 1) {
        const unsigned rx = (x & s) ? 1u : 0u, ry = (y & s) ? 1u : 0u;
        d += s * s * ((3u * rx) ^ ry);
        if (ry == 0) {
            if (rx == 1) { x = 65535u - x; y = 65535u - y; }
            std::swap(x, y);
        }
    }
    return d;
}

// Processing order of the velocities: along a Hilbert curve over the (vx, vy) plane, so that the
// velocities of a block are neighbours (their shifted windows overlap) and successive blocks touch
// neighbouring memory.  Ties and equal keys: by index.  The per-pixel result does not depend on it.
inline std::vector<std::pair<unsigned, int>> hilbert_order(const float* vel, int V) {
    float lox = vel[0], hix = vel[0], loy = vel[1], hiy = vel[1];
    for (int j = 1; j < V; ++j) {
        lox = std::min(lox, vel[2 * j]); hix = std::max(hix, vel[2 * j]);
        loy = std::min(loy, vel[2 * j + 1]); hiy = std::max(hiy, vel[2 * j + 1]);
    }
    const double ext = std::max({(double)hix - lox, (double)hiy - loy, 1e-30});
    std::vector<std::pair<unsigned, int>> key(V);
    for (int j = 0; j < V; ++j) {
        const unsigned qx = (unsigned)std::min(65535.0, ((double)vel[2 * j] - lox) / ext * 65535.0);
        const unsigned qy = (unsigned)std::min(65535.0, ((double)vel[2 * j + 1] - loy) / ext * 65535.0);
        key[j] = {hilbert_d(qx, qy), j};
    }
    std::sort(key.begin(), key.end());
    return key;
}

// Row pitch (in samples) of the encoded stack: W rounded up to even, so that every row starts
// 16-byte aligned and a pair of samples never straddles two rows.
__host__ __device__ constexpr int enc_pitch(int W) { return (W + 1) & ~1; }

// The encoded stack of the tiled and staged kernels: (psi, phi) -> (psi, -phi), invalid (psi NaN) ->
// (+0, +0); rows padded to Wp = enc_pitch(W) samples, the padding column is zero.  Adding a zero is
// exact, so one packed add per sample yields the in-order fp32 sums of both planes over the valid
// observations, and the sign bit of the second word is the validity flag.  One thread per pair.
__global__ void __launch_bounds__(256)
inline encode_kernel(const float2* __restrict__ in, float4* __restrict__ out, int W, int Wp, size_t rows) {
    const int half = Wp >> 1;
    const size_t total = rows * (size_t)half;
    const size_t stride = (size_t)gridDim.x * blockDim.x;
    for (size_t k = (size_t)blockIdx.x * blockDim.x + threadIdx.x; k < total; k += stride) {
        const size_t row = k / half;
        const int x = (int)(k - row * half) * 2;
        const float2* src = in + row * W + x;
        const float2 a = __ldg(src);
        const float2 b = (x + 1 < W) ? __ldg(src + 1) : make_float2(__int_as_float(0x7FC00000), 0.0f);
        const bool va = (a.x == a.x), vb = (b.x == b.x);
        float4 o;
        o.x = va ? a.x : 0.0f;
        o.y = va ? -a.y : 0.0f;
        o.z = vb ? b.x : 0.0f;
        o.w = vb ? -b.y : 0.0f;
        out[k] = o;
    }
}

}  // namespace kbmod

// One step S of the S5 pre-test / queue switch of the queued kernels (kernels 3 and 4): trajectory
// (velocity b_ = S / R, pixel r_ = S % R) is compacted into the warp's candidate queue if it is
// eligible and its approximate nu is not below the pixel's bound.  A step that fills the queue to 32
// leaves the switch (flush = true) so that one copy of the batch code serves all steps.  The kernel
// supplies VEL_OF(b) (velocity index of member b, < 0 = padding) and QPUT(qi, Psi, Phi, meta).
#define KBMOD_SCORE_STEP(S, VEL_OF, QPUT)                                                                \
    case S: {                                                                                            \
        constexpr int b_ = (S) / R, r_ = (S) % R;                                                        \
        const int j = VEL_OF(b_);                                                                        \
        if (j >= 0) {                                                                                    \
            const float Psi = __uint_as_float((unsigned)acc[b_][r_]);                                    \
            const float Phi = 0.0f - __uint_as_float((unsigned)(acc[b_][r_] >> 32));                     \
            unsigned n;                                                                                  \
            if constexpr (CM == 2) n = __popc(cnt[b_][r_ / RX] & ((r_ % RX) ? 0x55555555u : 0xAAAAAAAAu)); \
            else if constexpr (CM == 1) n = __popc(cnt[b_][r_ % NC]);                                    \
            else n = cnt[b_][r_ % NC];                                                                   \
            const bool pass = (n >= minobs) && (Phi > 0.0f) && ((inimg >> r_) & 1u) &&                   \
                              !(Psi * rsqrtf(Phi) < lo[r_]);                                             \
            const unsigned m = __ballot_sync(0xFFFFFFFFu, pass);                                         \
            if (m) {                                                                                     \
                if (pass) {                                                                              \
                    const unsigned qi = (qtail + __popc(m & ((1u << lane) - 1u))) & (QCAP - 1);          \
                    QPUT(qi, Psi, Phi, ((unsigned)j << 7) | (r_ << 5) | lane);                           \
                }                                                                                        \
                qtail += __popc(m);                                                                      \
                if (qtail - qhead >= 32) {                                                               \
                    step = (S) + 1;                                                                      \
                    flush = true;                                                                        \
                    break;                                                                               \
                }                                                                                        \
            }                                                                                            \
        }                                                                                                \
    }
#define KBMOD_SCORE_STEPS_32(VEL_OF, QPUT)                                                               \
    KBMOD_SCORE_STEP(0, VEL_OF, QPUT) KBMOD_SCORE_STEP(1, VEL_OF, QPUT) KBMOD_SCORE_STEP(2, VEL_OF, QPUT)    \
    KBMOD_SCORE_STEP(3, VEL_OF, QPUT) KBMOD_SCORE_STEP(4, VEL_OF, QPUT) KBMOD_SCORE_STEP(5, VEL_OF, QPUT)    \
    KBMOD_SCORE_STEP(6, VEL_OF, QPUT) KBMOD_SCORE_STEP(7, VEL_OF, QPUT) KBMOD_SCORE_STEP(8, VEL_OF, QPUT)    \
    KBMOD_SCORE_STEP(9, VEL_OF, QPUT) KBMOD_SCORE_STEP(10, VEL_OF, QPUT) KBMOD_SCORE_STEP(11, VEL_OF, QPUT)  \
    KBMOD_SCORE_STEP(12, VEL_OF, QPUT) KBMOD_SCORE_STEP(13, VEL_OF, QPUT) KBMOD_SCORE_STEP(14, VEL_OF, QPUT) \
    KBMOD_SCORE_STEP(15, VEL_OF, QPUT) KBMOD_SCORE_STEP(16, VEL_OF, QPUT) KBMOD_SCORE_STEP(17, VEL_OF, QPUT) \
    KBMOD_SCORE_STEP(18, VEL_OF, QPUT) KBMOD_SCORE_STEP(19, VEL_OF, QPUT) KBMOD_SCORE_STEP(20, VEL_OF, QPUT) \
    KBMOD_SCORE_STEP(21, VEL_OF, QPUT) KBMOD_SCORE_STEP(22, VEL_OF, QPUT) KBMOD_SCORE_STEP(23, VEL_OF, QPUT) \
    KBMOD_SCORE_STEP(24, VEL_OF, QPUT) KBMOD_SCORE_STEP(25, VEL_OF, QPUT) KBMOD_SCORE_STEP(26, VEL_OF, QPUT) \
    KBMOD_SCORE_STEP(27, VEL_OF, QPUT) KBMOD_SCORE_STEP(28, VEL_OF, QPUT) KBMOD_SCORE_STEP(29, VEL_OF, QPUT) \
    KBMOD_SCORE_STEP(30, VEL_OF, QPUT) KBMOD_SCORE_STEP(31, VEL_OF, QPUT)
