// search_staged.cu -- S3..S6, the fast path of kbmod_search (Eq.24-27).
//
// Design (B200-first; the paper's 32x16 thread blocks gathering through the cache, are prior art):
//   * S3 is hoisted to the host.  d = fl(v*dt_i) is uniform over start pixels, and for the
//     start pixels x0 = 0..W-1 the literal  floor(fl(fl(x0+d)+0.5f)) - x0  is piecewise constant
//     with breaks only where x0+d (or fl(x0+d)+0.5) crosses a power of two.  The host evaluates
//     the literal expression at every such break and proves, per (velocity, image, axis), that
//     one integer shift holds for the whole image; pairs it cannot prove take the literal
//     per-lane expression on the device.  The sampled pixels are identical to the definition.
//   * The stack is re-encoded once per call as (psi, -phi) with invalid samples = (+0,+0): one
//     packed add.rn.f32x2 accumulates both sums (adding zero is exact, so the result equals the
//     in-order fp32 sum over the valid observations), the sign bit of the second word is the
//     validity flag, and TMA's zero fill outside the image IS the "no observation" sample.
//   * A persistent CTA (one per SM) owns a 64x30 tile of start pixels at a time and walks the
//     velocity grid in blocks of B = 8 velocities that are neighbours in the (vx,vy) plane
//     (Hilbert order).  Every thread keeps Psi/Phi/validity history of 8 velocities x 4 pixels in
//     registers.  For each image the host has grouped the block's 8 shifted windows into
//     bounding boxes that fit a shared-memory slot; a producer warp streams these boxes with
//     cp.async.bulk.tensor (TMA, 3-D tensor map over [N][H][W], zero fill) into a ring of slots
//     guarded by full/empty mbarriers, and 15 consumer warps read them with conflict-free
//     LDS.64: 3 instructions per sample (LDS.64, FADD2, SHF).
//   * S5/S6: an approximate Psi*rsqrt(Phi) test against the pixel's current K-th best keeps
//     almost every trajectory off the exact path.  Survivors are compacted into a per-warp
//     queue; 32 at a time, one lane each, they are scored with correctly rounded sqrt/div and
//     inserted into the pixel's sorted list, which lives in the nu / vel_idx output planes.
//     Psi/Phi/n_obs/alpha of the K winners are re-evaluated literally at the end of the tile.
#include <algorithm>
#include <cmath>
#include <cstdlib>
#include <cstring>
#include <vector>

#include <cuda.h>

#include "ring_alloc.h"
#include "search_common.cuh"
#include "search_staged.cuh"
#include "topk_list.h"

namespace kbmod {

namespace {

// ---- geometry (compile-time)
constexpr int NCW = 15;                  // consumer warps (+ 1 producer warp = 512 threads, 128 registers each)
constexpr int RX = 2, RY = 2, R = RX * RY;   // pixels per thread: x = lane + 32*rx, y = 2*warp + ry
constexpr int TW = 32 * RX, TH = NCW * RY;   // start-pixel tile: 64 x 30
constexpr int THREADS = (NCW + 1) * 32;  // + 1 producer warp
constexpr int B = 8;                     // velocities per block
static_assert(B * R == 32, "the scoring switch of search_staged_kernel lists B*R = 32 steps");
// ring geometry variants (samples per slot, slots); selected per call by
// kbmod_search_options.staged_geom (tuning knob; default 0).  Smaller slots = more boxes in flight
// but fewer windows merged per box.
// Geometries 0-1: ring of equal slots (header + box): 4096 samples x 6 slots, 6144 x 4.
// Geometries 2-3: byte-granular data ring (ring_alloc.h) with a separate ring of VR_NH headers, so
// that the boxes in flight fill the whole shared memory whatever their sizes; cap = largest box
// (4096, 6144 samples).  The host plan's fill per sample byte at BASELINE.json configs[2] is 0.69
// with cap 4096 and 0.68 with cap 6144; smaller caps (2560, 3072: 0.72-0.78)
// and 8192 (0.69, fewer boxes in flight) were dropped in round 2.
constexpr int NGEOM = 4;
__host__ __device__ constexpr int cap_of(int g) { return (g == 0 || g == 2) ? 4096 : 6144; }
__host__ __device__ constexpr bool is_var(int g) { return g >= 2; }
constexpr int VR_NH = 16;                // header slots (= entries in flight at most) of the variable ring
constexpr int VR_RING_BYTES = 212992;    // data bytes of the variable ring (208 KB)
__host__ __device__ constexpr int nslot_of(int g) { return g == 0 ? 6 : g == 1 ? 4 : VR_NH; }
constexpr int HDR_INTS = 8 + 2 * B;
constexpr int HDR_BYTES = 128;
static_assert(HDR_INTS * 4 <= HDR_BYTES, "header");
__host__ __device__ constexpr int slot_bytes_of(int g) { return HDR_BYTES + cap_of(g) * 8; }
constexpr int QCAP = 64;                 // per-warp candidate queue entries
constexpr int MAXMAPS = 240;             // 240 x 128 B of tensor maps + the other parameters stay below the 32764-byte limit
constexpr int MAXBW = 128;               // box width limit (256 fp32 elements per TMA box row)
constexpr int SH_LIMIT = 30000;

// entry header (ints)
//  [0] type | flags << 8 | image << 16     [1] member mask      [2] row pitch of the box, bytes
//  [3] ox | oy << 16 (int16, box origin - tile origin)          [4] bw | bh << 16
//  [5] tensor-map id (ENT_TMA) / member b (ENT_UNSAFE)          [6],[7] vx, vy bits (ENT_UNSAFE);
//      on ENT_TMA entries the producer stores the box's byte offset in the data ring in [6]
//  [8 .. 8+B)    byte offset (from the box start) of member b's window origin
//  [8+B .. 8+2B) original velocity index of member b, -1 = padding (read on FLAG_LAST entries)
enum { ENT_NOP = 0, ENT_TMA = 1, ENT_UNSAFE = 2 };
enum { FLAG_LAST = 1, FLAG_EMPTY = 2 };

// shared memory: [ring][queues][full barriers][empty barriers][adv table]; ring = slots (fixed) or
// data bytes followed by the headers (variable)
__host__ __device__ constexpr size_t ring_bytes_of(int g) {
    return is_var(g) ? (size_t)VR_RING_BYTES + (size_t)VR_NH * HDR_BYTES : (size_t)nslot_of(g) * slot_bytes_of(g);
}
constexpr size_t smem_bytes_of(int g) {
    return ring_bytes_of(g) + (size_t)NCW * QCAP * 12 + 2 * nslot_of(g) * 8 + VR_NH * 4;
}
static_assert(smem_bytes_of(0) <= 227 * 1024 && smem_bytes_of(1) <= 227 * 1024 && smem_bytes_of(2) <= 227 * 1024 &&
              smem_bytes_of(3) <= 227 * 1024, "ring does not fit shared memory");
static_assert(cap_of(3) * 8 <= VR_RING_BYTES / 2, "a box must fit the variable ring comfortably");

// The literal S3 of include/kbmod_b200.h on the host (IEEE binary32, no contraction possible:
// two dependent additions).  d = fl(v*dt) is formed by the caller.
inline long long literal_offset(int x0, float d) {
    volatile float f = (float)x0 + d;
    volatile float g = f + 0.5f;
    return (long long)std::floor((double)g) - x0;
}

// Proves that floor(fl(fl(x0+d)+0.5f)) == x0 + s for every integer x0 in [0, n).  Between two
// consecutive breaks (x0+d or fl(x0+d)+0.5 crossing a power of two; |x0+d| <= 4 is checked
// point by point) both roundings act on x0-independent remainders, so the offset is constant:
// evaluating the literal expression on both sides of every break decides the whole range.
bool prove_shift(float d, int n, int& s) {
    const double dd = d;
    const long long s0 = literal_offset(0, d);
    auto same = [&](long long x0) {
        if (x0 < 0 || x0 >= n) return true;
        return literal_offset((int)x0, d) == s0;
    };
    if (!same(n - 1)) return false;
    for (int k = 2; k <= 16; ++k) {
        const double p = std::ldexp(1.0, k);
        for (int sg = -1; sg <= 1; sg += 2)
            for (int half = 0; half <= 1; ++half) {
                const double c = sg * p - 0.5 * half - dd;       // x0 + d = +-2^k (- 0.5)
                if (c < -3.0 || c > (double)n + 2.0) continue;
                const long long c0 = (long long)std::floor(c);
                for (long long x0 = c0 - 2; x0 <= c0 + 3; ++x0)
                    if (!same(x0)) return false;
            }
    }
    {
        const long long c0 = (long long)std::floor(-dd);
        for (long long x0 = c0 - 6; x0 <= c0 + 6; ++x0)
            if (!same(x0)) return false;
    }
    if (s0 < -SH_LIMIT || s0 > SH_LIMIT) return false;
    s = (int)s0;
    return true;
}

struct Group {
    unsigned mask;
    int sxlo, sxhi, sylo, syhi;
};
struct BoxQ { int qw, qh; };   // box-dimension quantisation (limits the number of tensor maps)

inline void box_of(const Group& g, const BoxQ& q, int& ox, int& bw, int& bh) {
    ox = g.sxlo & ~1;                               // 16-byte aligned box start (tile_x is even)
    bw = g.sxhi + TW - ox;
    bw = (bw + q.qw - 1) / q.qw * q.qw;
    bh = g.syhi - g.sylo + TH;
    bh = (bh + q.qh - 1) / q.qh * q.qh;
}
inline bool box_fits(int bw, int bh, int cap) { return bw <= MAXBW && bh <= 256 && bw * bh <= cap; }

}  // namespace

// Builds the entry stream.  Returns false when the box shapes cannot be brought under MAXMAPS.
static bool build_plan(const DtTable& dt, int N, int H, int W, const float* vel, int V, int cap, StagedPlan& plan) {
    plan.nent = 0;
    const std::vector<std::pair<unsigned, int>> key = hilbert_order(vel, V);    // processing order

    // proven shifts, per (velocity, image): 0 = skip (no observation possible), 1 = proven, 2 = unsafe
    std::vector<unsigned char> kind((size_t)V * N);
    std::vector<int> shx((size_t)V * N), shy((size_t)V * N);
    for (int j = 0; j < V; ++j)
        for (int i = 1; i < N; ++i) {
            volatile float dxf = vel[2 * j] * dt.dt[i];        // one fp32 multiply, as on the device
            volatile float dyf = vel[2 * j + 1] * dt.dt[i];
            const float dx = dxf, dy = dyf;
            unsigned char k;
            int sx = 0, sy = 0;
            if (!(std::fabs(dx) < (float)SH_LIMIT && std::fabs(dy) < (float)SH_LIMIT)) k = 0;
            else k = (prove_shift(dx, W, sx) && prove_shift(dy, H, sy)) ? 1 : 2;
            kind[(size_t)j * N + i] = k;
            shx[(size_t)j * N + i] = sx;
            shy[(size_t)j * N + i] = sy;
        }

    const int nblk = (V + B - 1) / B;
    static const BoxQ levels[] = {{2, 1}, {2, 2}, {4, 2}, {4, 4}, {8, 4}, {8, 8}, {16, 8}, {16, 16}, {32, 32}};
    for (const BoxQ& q : levels) {
        plan.stream.clear();
        plan.shapes.clear();
        bool too_many = false;
        for (int blk = 0; blk < nblk && !too_many; ++blk) {
            int jb[B];
            for (int b = 0; b < B; ++b) jb[b] = (blk * B + b < V) ? key[blk * B + b].second : -1;
            const size_t first = plan.stream.size();
            auto new_entry = [&](int type, int img) -> int* {
                plan.stream.resize(plan.stream.size() + HDR_INTS, 0);
                int* e = plan.stream.data() + plan.stream.size() - HDR_INTS;
                e[0] = type | (img << 16);
                for (int b = 0; b < B; ++b) e[8 + B + b] = jb[b];
                return e;
            };
            for (int i = 1; i < N; ++i) {
                std::vector<Group> groups;
                for (int b = 0; b < B; ++b) {
                    if (jb[b] < 0) continue;
                    const size_t k = (size_t)jb[b] * N + i;
                    if (kind[k] == 1) groups.push_back({1u << b, shx[k], shx[k], shy[k], shy[k]});
                    else if (kind[k] == 2) {
                        int* e = new_entry(ENT_UNSAFE, i);
                        e[5] = b;
                        std::memcpy(&e[6], &vel[2 * jb[b]], 4);
                        std::memcpy(&e[7], &vel[2 * jb[b] + 1], 4);
                    }
                }
                // greedy agglomeration: merge the pair that saves the most box area while it fits
                for (;;) {
                    int ba = -1, bc = -1, best = 0;
                    for (size_t a = 0; a < groups.size(); ++a)
                        for (size_t c = a + 1; c < groups.size(); ++c) {
                            Group m{groups[a].mask | groups[c].mask, std::min(groups[a].sxlo, groups[c].sxlo),
                                    std::max(groups[a].sxhi, groups[c].sxhi), std::min(groups[a].sylo, groups[c].sylo),
                                    std::max(groups[a].syhi, groups[c].syhi)};
                            int ox, bw, bh, wa, ha, wc, hc;
                            box_of(m, q, ox, bw, bh);
                            if (!box_fits(bw, bh, cap)) continue;
                            box_of(groups[a], q, ox, wa, ha);
                            box_of(groups[c], q, ox, wc, hc);
                            const int save = wa * ha + wc * hc - bw * bh;
                            if (save > best) { best = save; ba = (int)a; bc = (int)c; }
                        }
                    if (ba < 0) break;
                    Group& ga = groups[ba];
                    const Group& gc = groups[bc];
                    ga = {ga.mask | gc.mask, std::min(ga.sxlo, gc.sxlo), std::max(ga.sxhi, gc.sxhi),
                          std::min(ga.sylo, gc.sylo), std::max(ga.syhi, gc.syhi)};
                    groups.erase(groups.begin() + bc);
                }
                for (const Group& g : groups) {
                    int ox, bw, bh;
                    box_of(g, q, ox, bw, bh);
                    if (!box_fits(bw, bh, cap)) { too_many = true; break; }   // quantised singleton too big
                    int id = -1;
                    for (size_t m = 0; m < plan.shapes.size(); ++m)
                        if (plan.shapes[m].first == bw && plan.shapes[m].second == bh) { id = (int)m; break; }
                    if (id < 0) {
                        if ((int)plan.shapes.size() >= MAXMAPS) { too_many = true; break; }
                        id = (int)plan.shapes.size();
                        plan.shapes.push_back({bw, bh});
                    }
                    int* e = new_entry(ENT_TMA, i);
                    e[1] = (int)g.mask;
                    e[2] = bw * 8;
                    e[3] = (int)(((unsigned)g.sylo << 16) | ((unsigned)ox & 0xFFFFu));
                    e[4] = bw | (bh << 16);
                    e[5] = id;
                    for (int b = 0; b < B; ++b)
                        if (g.mask & (1u << b)) {
                            const size_t k = (size_t)jb[b] * N + i;
                            e[8 + b] = ((shy[k] - g.sylo) * bw + (shx[k] - ox)) * 8;
                        }
                }
                if (too_many) break;
            }
            if (too_many) break;
            if (plan.stream.size() == first) new_entry(ENT_NOP, 0);
            plan.stream[plan.stream.size() - HDR_INTS] |= FLAG_LAST << 8;
        }
        if (!too_many) {
            plan.nent = (int)(plan.stream.size() / HDR_INTS);
            return true;
        }
    }
    return false;
}

size_t staged_plan_bytes(int N, int V) {
    const size_t nblk = ((size_t)V + B - 1) / B;
    return nblk * ((size_t)std::max(N - 1, 0) * B + 1) * HDR_INTS * sizeof(int) + 256;
}
size_t staged_enc_bytes(int N, int H, int W) { return (size_t)N * H * enc_pitch(W) * sizeof(float2); }

int staged_plan_build(const DtTable& dt, int N, int H, int W, const float* vel_host, int V, int geom,
                      StagedPlan& plan) {
    // limits of the int16 shift encoding, the queue's 24-bit velocity index, the TMA coordinates
    if (W > SH_LIMIT || H > SH_LIMIT || V >= (1 << 24)) return KBMOD_ERR_UNSUPPORTED;
    if (geom < 0 || geom >= NGEOM) return KBMOD_ERR_ARG;
    plan.geom = geom;
    if (!build_plan(dt, N, H, W, vel_host, V, cap_of(geom), plan)) return KBMOD_ERR_UNSUPPORTED;
    if (plan.stream.size() * sizeof(int) > staged_plan_bytes(N, V)) return KBMOD_ERR_UNSUPPORTED;
    return KBMOD_OK;
}

int staged_plan_debug(const DtTable& dt, int N, int H, int W, const float* vel_host, int V, int geom,
                      int32_t* stream, size_t stream_ints, int32_t* shapes, int max_shapes, int32_t* info) {
    StagedPlan plan;
    if (int rc = staged_plan_build(dt, N, H, W, vel_host, V, geom, plan)) return rc;
    const int cap = cap_of(geom);
    info[0] = plan.nent; info[1] = HDR_INTS; info[2] = (int)plan.shapes.size(); info[3] = TW;
    info[4] = TH; info[5] = B; info[6] = cap; info[7] = HDR_BYTES;
    if (plan.stream.size() > stream_ints || (int)plan.shapes.size() > max_shapes) return KBMOD_ERR_WORKSPACE;
    std::memcpy(stream, plan.stream.data(), plan.stream.size() * sizeof(int));
    for (size_t m = 0; m < plan.shapes.size(); ++m) {
        shapes[2 * m] = plan.shapes[m].first;
        shapes[2 * m + 1] = plan.shapes[m].second;
    }
    return KBMOD_OK;
}

// ---------------------------------------------------------------------------------------------
// device side
// ---------------------------------------------------------------------------------------------
typedef unsigned long long u64;

// The inline-PTX helpers.  tests/test_staged_simt.py compiles this file with g++ against a SIMT
// emulator (tests/hostlogic/simt/) and defines KBMOD_SIMT_EMUL as the header that supplies host
// stand-ins of the same names; the product build never defines it.
#if defined(KBMOD_SIMT_EMUL)
#include KBMOD_SIMT_EMUL
#else
__device__ __forceinline__ unsigned smem_u32(const void* p) { return (unsigned)__cvta_generic_to_shared(p); }
__device__ __forceinline__ void mbar_init(unsigned bar, unsigned count) {
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(bar), "r"(count) : "memory");
}
__device__ __forceinline__ void fence_mbar_init() {
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
}
__device__ __forceinline__ void mbar_arrive(unsigned bar) {
    asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];" ::"r"(bar) : "memory");
}
__device__ __forceinline__ void mbar_arrive_expect_tx(unsigned bar, unsigned bytes) {
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(bar), "r"(bytes) : "memory");
}
__device__ __forceinline__ bool mbar_try_wait(unsigned bar, unsigned parity) {
    unsigned ok;
    asm volatile(
        "{\n"
        ".reg .pred p;\n"
        "mbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2;\n"
        "selp.u32 %0, 1, 0, p;\n"
        "}\n" : "=r"(ok) : "r"(bar), "r"(parity) : "memory");
    return ok != 0;
}
__device__ __forceinline__ void tma_load_3d(unsigned dst, const void* tmap, int c0, int c1, int c2, unsigned bar) {
    asm volatile(
        "cp.async.bulk.tensor.3d.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1, {%2, %3, %4}], [%5];"
        ::"r"(dst), "l"(tmap), "r"(c0), "r"(c1), "r"(c2), "r"(bar) : "memory");
}
template <int OFF>
__device__ __forceinline__ u64 lds64(unsigned a) {
    u64 v;
    asm volatile("ld.shared.b64 %0, [%1+%2];" : "=l"(v) : "r"(a), "n"(OFF));
    return v;
}
__device__ __forceinline__ void sts32(unsigned a, int v) {
    asm volatile("st.shared.b32 [%0], %1;" ::"r"(a), "r"(v) : "memory");
}
__device__ __forceinline__ int lds32(unsigned a) {
    int v;
    asm volatile("ld.shared.b32 %0, [%1];" : "=r"(v) : "r"(a));
    return v;
}
__device__ __forceinline__ int4 lds128(unsigned a) {
    int4 v;
    asm volatile("ld.shared.v4.b32 {%0,%1,%2,%3}, [%4];" : "=r"(v.x), "=r"(v.y), "=r"(v.z), "=r"(v.w) : "r"(a));
    return v;
}
#endif  // KBMOD_SIMT_EMUL

// Warp-uniform bounded wait (all 32 lanes must call it).  A wait that lasts WAIT_LIMIT_CLOCKS
// (about two seconds; a healthy wait is microseconds) means the pipeline is broken: the warp
// gives up instead of hanging the GPU, and the caller reports KBMOD_ERR_TIMEOUT.
constexpr long long WAIT_LIMIT_CLOCKS = 1ll << 32;
__device__ __forceinline__ bool mbar_wait(unsigned bar, unsigned parity) {
    bool ok = mbar_try_wait(bar, parity);
    if (!ok) {
        const long long t0 = clock64();
        for (;;) {
            ok = mbar_try_wait(bar, parity);
            if (ok || clock64() - t0 > WAIT_LIMIT_CLOCKS) break;
        }
    }
    return __all_sync(0xFFFFFFFFu, ok);
}
__device__ __forceinline__ void acc_add(u64& a, u64 s) {      // (Psi, -Phi) += (psi, -phi), RN each
    float2 fa = make_float2(__uint_as_float((unsigned)a), __uint_as_float((unsigned)(a >> 32)));
    float2 fs = make_float2(__uint_as_float((unsigned)s), __uint_as_float((unsigned)(s >> 32)));
    fa = __fadd2_rn(fa, fs);
    a = (u64)__float_as_uint(fa.x) | ((u64)__float_as_uint(fa.y) << 32);
}
struct StagedMaps { CUtensorMap m[MAXMAPS]; };

struct StagedParams {
    const float2* psiphi;     // original stack (final re-evaluation of the winners)
    const u64* enc;           // encoded stack, row pitch Wp
    const int* plan;          // nent entries of HDR_INTS ints
    const float2* vel;        // caller's velocity table (device copy)
    int* status;              // device word: set to 1 by a warp whose barrier wait timed out
    int nent, N, H, W, Wp, K, min_obs;
    int y_begin, y_end;       // band of start rows; the result planes hold rows y_begin..y_end-1 only
    int tiles_x, tiles_y, ntiles, group_w;
    kbmod_result out;
    DtTable dt;
};

__device__ __forceinline__ void tile_of(const StagedParams& prm, int t, int& tile_x, int& tile_y) {
    // groups of group_w tile columns, row-major inside a group: the tiles being worked on at the
    // same time cover a compact region, so their windows share L2 lines
    const int per_group = prm.group_w * prm.tiles_y;
    const int g = t / per_group, rem = t - g * per_group;
    const int gw = min(prm.group_w, prm.tiles_x - g * prm.group_w);
    const int ty = rem / gw;
    const int tx = g * prm.group_w + (rem - ty * gw);
    tile_x = tx * TW;
    tile_y = prm.y_begin + ty * TH;
}

// memory policy of the per-pixel lists: they live in the nu / vel_idx output planes and are read
// and written through L2 (only the owning warp touches a pixel's list)
struct ListMemL2 {
    template <class T> static __device__ __forceinline__ T ld(const T* p) { return __ldcg(p); }
    template <class T> static __device__ __forceinline__ void st(T* p, T v) { __stcg(p, v); }
};

// One dense pass over up to 32 queued candidates of this warp: lane l takes entry qhead + l.
template <int KP>
__device__ __forceinline__ void process_batch(const StagedParams& prm, unsigned qb, unsigned qhead, int n, int lane,
                                              int wx0, int wy0) {
    bool valid = lane < n;
    const unsigned idx = (qhead + lane) & (QCAP - 1);
    const float Psi = __int_as_float(lds32(qb + 4 * idx));
    const float Phi = __int_as_float(lds32(qb + 4 * QCAP + 4 * idx));
    const unsigned meta = (unsigned)lds32(qb + 8 * QCAP + 4 * idx);
    const int pix = meta & 127, j = (int)(meta >> 7);
    const int r = pix >> 5, ln = pix & 31;
    const int x = wx0 + ln + 32 * (r % RX), y = wy0 + r / RX;
    const float nu = valid ? score_nu(Psi, Phi) : 0.0f;
    const size_t p = valid ? ((size_t)(y - prm.y_begin) * prm.W + x) * prm.K : 0;
    for (;;) {
        // two candidates of the same pixel in one batch: lowest lane first, the rest next round
        const unsigned same = __match_any_sync(0xFFFFFFFFu, valid ? pix : 128 + lane);
        if (valid && lane == __ffs(same) - 1) {
            list_insert<KP, ListMemL2>(prm.out.nu + p, prm.out.vel_idx + p, prm.K, nu, j);
            valid = false;
        }
        __syncwarp();
        if (!__any_sync(0xFFFFFFFFu, valid)) break;
    }
}

// literal S3 + S4 of one trajectory on the original stack (winners' re-evaluation)
__device__ __forceinline__ void coadd_literal(const StagedParams& prm, int x0, int y0, float2 v, float& Psi,
                                              float& Phi, int& n) {
    Psi = 0.0f; Phi = 0.0f; n = 0;
    for (int i = 0; i < prm.N; ++i) {
        int ix, iy;
        if (traj_pixel(x0, v.x, prm.dt.dt[i], prm.W, ix) && traj_pixel(y0, v.y, prm.dt.dt[i], prm.H, iy)) {
            const float2 s = __ldg(prm.psiphi + ((size_t)i * prm.H + iy) * prm.W + ix);
            if (s.x == s.x) { Psi = __fadd_rn(Psi, s.x); Phi = __fadd_rn(Phi, s.y); ++n; }
        }
    }
}

static_assert(sizeof(StagedParams) + sizeof(StagedMaps) <= 32764, "kernel parameters exceed the 32764-byte limit");

// CM: how the validity of the samples is counted.  2: history bits, the two rx pixels of a row
// share a register (N <= 16); 1: history bits, one register per pixel (N <= 32); 0: additive.
template <int CM, int KP, int G>
__global__ void __launch_bounds__(THREADS, 1)
search_staged_kernel(const __grid_constant__ StagedParams prm, const __grid_constant__ StagedMaps maps) {
    constexpr bool VR = is_var(G);                    // byte-granular data ring + header ring
    constexpr int NSLOT = nslot_of(G), SLOT_BYTES = slot_bytes_of(G);
    extern __shared__ __align__(128) unsigned char smem_raw[];
    const unsigned ring = smem_u32(smem_raw);
    const unsigned hdrs = ring + VR_RING_BYTES;       // VR only: NSLOT headers of HDR_BYTES
    const unsigned qall = ring + (unsigned)ring_bytes_of(G);
    const unsigned bar_full = qall + NCW * QCAP * 12;
    const unsigned bar_empty = bar_full + NSLOT * 8;
    // header and box of ring slot s (fixed geometry: the box follows its header; variable: the
    // box sits in the data ring at the offset the producer stored in header int 6)
    auto hdr_of = [&](unsigned s) -> unsigned { return VR ? hdrs + s * HDR_BYTES : ring + s * SLOT_BYTES; };
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const int N = prm.N, H = prm.H, W = prm.W, K = prm.K;

    if (tid == 0) {
        for (int s = 0; s < NSLOT; ++s) {
            mbar_init(bar_full + 8 * s, 1);
            mbar_init(bar_empty + 8 * s, NCW);
        }
        fence_mbar_init();
    }
    __syncthreads();

    const int my_tiles = ((int)blockIdx.x < prm.ntiles) ? (prm.ntiles - (int)blockIdx.x + (int)gridDim.x - 1) / (int)gridDim.x : 0;

    if (warp == NCW) {
        // ================= producer warp: header + TMA box per entry =================
        constexpr int PF = 4;                       // header prefetch distance (entries)
        const long long total = (long long)my_tiles * prm.nent;
        int hreg[PF];
#pragma unroll
        for (int p = 0; p < PF; ++p)
            hreg[p] = (p < total && lane < HDR_INTS) ? __ldg(prm.plan + (size_t)(p % prm.nent) * HDR_INTS + lane) : 0;
        int e = 0, k = 0, tile_x = 0, tile_y = 0;
        if (my_tiles > 0) tile_of(prm, blockIdx.x, tile_x, tile_y);
        unsigned slot = 0, use = 0;
        // VR: allocator state (identical in all lanes; adv[] in shared memory) and the ring slot /
        // phase of the oldest entry not yet released
        RingAlloc<VR_RING_BYTES, VR_NH> ra(reinterpret_cast<unsigned*>(smem_raw + (bar_empty - ring) + NSLOT * 8));
        unsigned oslot = 0, ophase = 0;
        for (long long g0 = 0; g0 < total; g0 += PF) {
#pragma unroll
            for (int p = 0; p < PF; ++p) {
                const long long g = g0 + p;
                if (g < total) {
                    int hv = hreg[p];
                    if (g + PF < total && lane < HDR_INTS)
                        hreg[p] = __ldg(prm.plan + (size_t)((e + PF) % prm.nent) * HDR_INTS + lane);
                    const int h0 = __shfl_sync(0xFFFFFFFFu, hv, 0), h3 = __shfl_sync(0xFFFFFFFFu, hv, 3);
                    const int h4 = __shfl_sync(0xFFFFFFFFu, hv, 4), h5 = __shfl_sync(0xFFFFFFFFu, hv, 5);
                    const int type = h0 & 0xFF, img = h0 >> 16;
                    const int bw = h4 & 0xFFFF, bh = h4 >> 16;
                    const int gx = tile_x + (short)(h3 & 0xFFFF), gy = tile_y + (h3 >> 16);
                    const bool load = (type == ENT_TMA) && !(gx + bw <= 0 || gx >= W || gy + bh <= 0 || gy >= H);
                    if (type == ENT_TMA && !load && lane == 0) hv |= FLAG_EMPTY << 8;
                    const unsigned sa = hdr_of(slot);
                    unsigned box_at;
                    if constexpr (VR) {
                        // place the box in the data ring; release finished entries (in order) until it fits
                        const unsigned need = load ? (((unsigned)(bw * bh * 8) + 127u) & ~127u) : 0u;
                        while (!ra.fits(need)) {
                            if (!mbar_wait(bar_empty + 8 * oslot, ophase)) {
                                if (lane == 0) atomicExch(prm.status, 1);
                                return;
                            }
                            ra.release_oldest();
                            if (++oslot == NSLOT) { oslot = 0; ophase ^= 1; }
                        }
                        // adv[] is shared by the 32 lanes: when the header ring is the limit, place()
                        // rewrites the very word release_oldest() has just read (next % NH == oldest %
                        // NH), so no lane may place before every lane has released (found by the SIMT
                        // emulation, tests/test_staged_simt.py: lanes are not in lockstep)
                        __syncwarp();
                        const unsigned off = ra.place(need);
                        box_at = ring + off;
                        if (type == ENT_TMA && lane == 6) hv = (int)off;
                    } else {
                        if (use > 0 && !mbar_wait(bar_empty + 8 * slot, (use - 1) & 1)) {
                            if (lane == 0) atomicExch(prm.status, 1);
                            return;
                        }
                        box_at = sa + HDR_BYTES;
                        if (type == ENT_TMA && lane == 6) hv = HDR_BYTES + (int)(slot * SLOT_BYTES);
                    }
                    if (lane < HDR_INTS) sts32(sa + 4 * lane, hv);
                    __syncwarp();
                    if (lane == 0) {
                        if (load) {
                            mbar_arrive_expect_tx(bar_full + 8 * slot, (unsigned)(bw * bh * 8));
                            tma_load_3d(box_at, &maps.m[h5], 2 * gx, gy, img, bar_full + 8 * slot);
                        } else {
                            mbar_arrive(bar_full + 8 * slot);
                        }
                    }
                    if (++slot == NSLOT) { slot = 0; ++use; }
                    if (++e == prm.nent) {
                        e = 0;
                        if (++k < my_tiles) tile_of(prm, blockIdx.x + k * gridDim.x, tile_x, tile_y);
                    }
                }
            }
        }
        return;
    }

    // ================= consumer warps =================
    constexpr int NC = (CM == 2) ? RY : R;        // count registers per velocity
    const unsigned qb = qall + warp * (QCAP * 12);
    unsigned slot = 0, phase = 0;
    const unsigned minobs = (unsigned)prm.min_obs;

    for (int kt = 0; kt < my_tiles; ++kt) {
        int tile_x, tile_y;
        tile_of(prm, blockIdx.x + kt * gridDim.x, tile_x, tile_y);
        const int x_first = tile_x + lane, y_first = tile_y + warp * RY;
        unsigned inimg = 0;                        // bit r: pixel r of this thread is a start pixel of the band
#pragma unroll
        for (int r = 0; r < R; ++r)
            inimg |= ((x_first + 32 * (r % RX) < W) && (y_first + r / RX < prm.y_end)) ? (1u << r) : 0u;
        // result-plane position (band-relative rows) of pixel r: pix0 + 32*rx + ry*W
        const size_t pix0 = (size_t)(y_first - prm.y_begin) * W + x_first;
        const u64* enc0 = prm.enc + (size_t)y_first * prm.Wp + x_first;  // image 0 samples of this thread

        // empty lists
#pragma unroll
        for (int r = 0; r < R; ++r)
            if (inimg & (1u << r)) {
                const size_t p = (pix0 + 32 * (r % RX) + (size_t)(r / RX) * W) * K;
                for (int kk = 0; kk < K; ++kk) {
                    __stcg(prm.out.nu + p + kk, -INFINITY);
                    __stcg(prm.out.vel_idx + p + kk, LIST_EMPTY_IDX);
                }
            }
        __syncwarp();
        unsigned qhead = 0, qtail = 0;

        u64 acc[B][R];
        unsigned cnt[B][NC];
        float lo[R];                               // pre-test bound: K-th best nu minus a safety margin
        bool fresh = true;                         // next entry starts a velocity block

        for (int e = 0; e < prm.nent; ++e) {
            if (fresh) {
                fresh = false;
                // image 0 (dt = 0: shift (0,0) for every velocity) initialises the sums
                u64 s0[R];
#pragma unroll
                for (int r = 0; r < R; ++r)
                    s0[r] = (inimg & (1u << r)) ? __ldg(enc0 + 32 * (r % RX) + (size_t)(r / RX) * prm.Wp) : 0ull;
#pragma unroll
                for (int b = 0; b < B; ++b) {
#pragma unroll
                    for (int r = 0; r < R; ++r) acc[b][r] = s0[r];
                    if constexpr (CM == 2) {
#pragma unroll
                        for (int ry = 0; ry < RY; ++ry)
                            cnt[b][ry] = (unsigned)(s0[ry * RX] >> 63) * 2u + (unsigned)(s0[ry * RX + 1] >> 63);
                    } else {
#pragma unroll
                        for (int r = 0; r < R; ++r) cnt[b][r] = (unsigned)(s0[r] >> 63);
                    }
                }
#pragma unroll
                for (int r = 0; r < R; ++r) {
                    float w = -INFINITY;
                    if (inimg & (1u << r))
                        w = __ldcg(prm.out.nu + (pix0 + 32 * (r % RX) + (size_t)(r / RX) * W) * K + (K - 1));
                    lo[r] = fmaf(-fabsf(w), 4e-6f, w);                   // -inf stays -inf
                }
            }

            const unsigned sa = hdr_of(slot);
            if (!mbar_wait(bar_full + 8 * slot, phase)) {
                if (lane == 0) atomicExch(prm.status, 1);
                return;
            }
            const int4 h = lds128(sa);
            const int type = h.x & 0xFF, flags = (h.x >> 8) & 0xFF;
            if (type == ENT_TMA && !(flags & FLAG_EMPTY)) {
                const unsigned pitch = (unsigned)h.z;
                // header int 6 = byte offset of the box from the start of the ring (both geometries)
                const unsigned thr = ring + (unsigned)lds32(sa + 24) + lane * 8 + (unsigned)(warp * RY) * pitch;
#pragma unroll
                for (int b = 0; b < B; ++b) {
                    if (h.y & (1 << b)) {
                        unsigned a = thr + (unsigned)lds32(sa + 32 + 4 * b);
#pragma unroll
                        for (int ry = 0; ry < RY; ++ry) {
                            const u64 sA = lds64<0>(a), sB = lds64<256>(a);
                            acc_add(acc[b][ry * RX], sA);
                            acc_add(acc[b][ry * RX + 1], sB);
                            if constexpr (CM == 2) {
                                cnt[b][ry] = __funnelshift_l((unsigned)(sA >> 32), cnt[b][ry], 1);
                                cnt[b][ry] = __funnelshift_l((unsigned)(sB >> 32), cnt[b][ry], 1);
                            } else if constexpr (CM == 1) {
                                cnt[b][ry * RX] = __funnelshift_l((unsigned)(sA >> 32), cnt[b][ry * RX], 1);
                                cnt[b][ry * RX + 1] = __funnelshift_l((unsigned)(sB >> 32), cnt[b][ry * RX + 1], 1);
                            } else {
                                cnt[b][ry * RX] += (unsigned)(sA >> 63);
                                cnt[b][ry * RX + 1] += (unsigned)(sB >> 63);
                            }
                            a += pitch;
                        }
                    }
                }
            } else if (type == ENT_UNSAFE) {
                // shift not proven for this (velocity, image): the literal per-lane S3
                const int4 h1 = lds128(sa + 16);
                const int bsel = h1.y, img = h.x >> 16;
                const float vx = __int_as_float(h1.z), vy = __int_as_float(h1.w), dti = prm.dt.dt[img];
                u64 s[R];
#pragma unroll
                for (int ry = 0; ry < RY; ++ry) {
                    int y = 0;
                    const bool yin = traj_pixel(y_first + ry, vy, dti, H, y);
#pragma unroll
                    for (int rx = 0; rx < RX; ++rx) {
                        int x = 0;
                        const bool in = traj_pixel(x_first + 32 * rx, vx, dti, W, x) && yin;
                        s[ry * RX + rx] = in ? __ldg(prm.enc + ((size_t)img * H + y) * prm.Wp + x) : 0ull;
                    }
                }
#pragma unroll
                for (int b = 0; b < B; ++b)
                    if (b == bsel) {
#pragma unroll
                        for (int r = 0; r < R; ++r) {
                            acc_add(acc[b][r], s[r]);
                            if constexpr (CM == 2) cnt[b][r / RX] = __funnelshift_l((unsigned)(s[r] >> 32), cnt[b][r / RX], 1);
                            else if constexpr (CM == 1) cnt[b][r] = __funnelshift_l((unsigned)(s[r] >> 32), cnt[b][r], 1);
                            else cnt[b][r] += (unsigned)(s[r] >> 63);
                        }
                    }
            }

            if (flags & FLAG_LAST) {
                // ---- S5 + S6 for the B x R trajectories of this block.  The steps are the cases of
                // one switch so that a single copy of the batch code serves all of them: a step that
                // fills the queue to 32 leaves the switch, the batch is processed, and the switch is
                // re-entered at the next step.
                fresh = true;
                int step = 0;
                for (;;) {
                    bool flush = false;
                    switch (step) {
#define KBMOD_VEL_OF(b) lds32(sa + 32 + 4 * B + 4 * (b))
#define KBMOD_QPUT(qi, Psi, Phi, meta)                                                       \
    (sts32(qb + 4 * (qi), __float_as_int(Psi)), sts32(qb + 4 * QCAP + 4 * (qi), __float_as_int(Phi)), \
     sts32(qb + 8 * QCAP + 4 * (qi), (int)(meta)))
                        KBMOD_SCORE_STEPS_32(KBMOD_VEL_OF, KBMOD_QPUT)
#undef KBMOD_VEL_OF
#undef KBMOD_QPUT
                        default: break;
                    }
                    if (!flush) break;
                    __syncwarp();
                    process_batch<KP>(prm, qb, qhead, 32, lane, tile_x, y_first);
                    qhead += 32;
                }
            }
            __syncwarp();
            if (lane == 0) mbar_arrive(bar_empty + 8 * slot);
            if (++slot == NSLOT) { slot = 0; phase ^= 1; }
        }

        // ---- end of tile: drain the queue, then re-evaluate the winners literally and write them
        while (qtail != qhead) {
            const int n = min(32u, qtail - qhead);
            process_batch<KP>(prm, qb, qhead, n, lane, tile_x, y_first);
            qhead += n;
        }
        __syncwarp();
#pragma unroll 1
        for (int r = 0; r < R; ++r) {
            if (!(inimg & (1u << r))) continue;
            const int x0 = x_first + 32 * (r % RX), y0 = y_first + r / RX;
            const size_t p = ((size_t)(y0 - prm.y_begin) * W + x0) * K;
            for (int kk = 0; kk < K; ++kk) {
                const int j = __ldcg(prm.out.vel_idx + p + kk);
                if (j != LIST_EMPTY_IDX) {
                    float Psi, Phi;
                    int n;
                    coadd_literal(prm, x0, y0, __ldg(prm.vel + j), Psi, Phi, n);
                    prm.out.n_obs[p + kk] = n;
                    prm.out.psi[p + kk] = Psi;
                    prm.out.phi[p + kk] = Phi;
                    prm.out.nu[p + kk] = score_nu(Psi, Phi);
                    prm.out.alpha[p + kk] = score_alpha(Psi, Phi);
                } else {
                    prm.out.vel_idx[p + kk] = -1;
                    prm.out.n_obs[p + kk] = 0;
                    prm.out.psi[p + kk] = 0.0f;
                    prm.out.phi[p + kk] = 0.0f;
                    prm.out.nu[p + kk] = -INFINITY;
                    prm.out.alpha[p + kk] = 0.0f;
                }
            }
        }
    }
}

// ---------------------------------------------------------------------------------------------
// launch
// ---------------------------------------------------------------------------------------------
typedef CUresult (*EncodeTiledFn)(CUtensorMap*, CUtensorMapDataType, cuuint32_t, void*, const cuuint64_t*,
                                  const cuuint64_t*, const cuuint32_t*, const cuuint32_t*, CUtensorMapInterleave,
                                  CUtensorMapSwizzle, CUtensorMapL2promotion, CUtensorMapFloatOOBfill);

static EncodeTiledFn encode_tiled_fn() {
    static EncodeTiledFn fn = [] {
        void* p = nullptr;
        cudaDriverEntryPointQueryResult qr;
        if (cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &p, cudaEnableDefault, &qr) != cudaSuccess ||
            qr != cudaDriverEntryPointSuccess)
            p = nullptr;
        return (EncodeTiledFn)p;
    }();
    return fn;
}

template <int CM, int KP, int G>
static int launch_variant(const StagedParams& prm, const StagedMaps& maps, int grid, cudaStream_t st) {
    auto kern = search_staged_kernel<CM, KP, G>;
    // per launch, not cached: the attribute belongs to the current device's copy of the function
    if (cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem_bytes_of(G)) != cudaSuccess)
        return KBMOD_ERR_CUDA;
    KBMOD_LAUNCH(kern, grid, THREADS, smem_bytes_of(G), st, prm, maps);
    note_launch();
    return cudaGetLastError() == cudaSuccess ? KBMOD_OK : KBMOD_ERR_CUDA;
}
template <int CM, int KP>
static int launch_geom(int g, const StagedParams& prm, const StagedMaps& maps, int grid, cudaStream_t st) {
    switch (g) {
        case 1: return launch_variant<CM, KP, 1>(prm, maps, grid, st);
        case 2: return launch_variant<CM, KP, 2>(prm, maps, grid, st);
        case 3: return launch_variant<CM, KP, 3>(prm, maps, grid, st);
        default: return launch_variant<CM, KP, 0>(prm, maps, grid, st);
    }
}

int staged_launch(const StagedPlan& plan, const float2* psiphi, const DtTable& dt, int N, int H, int W, int K,
                  int min_obs, int y_begin, int y_end, const kbmod_result& out, void* plan_dev,
                  const float2* vel_dev, float2* enc_dev, int* status_dev, cudaStream_t st) {
    EncodeTiledFn enc_fn = encode_tiled_fn();
    if (!enc_fn) return KBMOD_ERR_UNSUPPORTED;
    const int geom = plan.geom;
    if (cudaMemcpyAsync(plan_dev, plan.stream.data(), plan.stream.size() * sizeof(int), cudaMemcpyHostToDevice, st) != cudaSuccess)
        return KBMOD_ERR_CUDA;

    if (cudaMemsetAsync(status_dev, 0, sizeof(int), st) != cudaSuccess) return KBMOD_ERR_CUDA;
    const int Wp = enc_pitch(W);
    KBMOD_LAUNCH(encode_kernel, 148 * 8, 256, 0, st, psiphi, reinterpret_cast<float4*>(enc_dev), W, Wp, (size_t)N * H);
    note_launch();
    if (cudaGetLastError() != cudaSuccess) return KBMOD_ERR_CUDA;

    // one 3-D tensor map (x: 2*Wp floats, y: H, image: N) per distinct box shape; zero fill outside
    StagedMaps maps;
    std::memset(&maps, 0, sizeof(maps));
    for (size_t m = 0; m < plan.shapes.size(); ++m) {
        cuuint64_t dims[3] = {(cuuint64_t)2 * Wp, (cuuint64_t)H, (cuuint64_t)N};
        cuuint64_t strides[2] = {(cuuint64_t)Wp * 8, (cuuint64_t)Wp * 8 * H};
        cuuint32_t box[3] = {(cuuint32_t)(2 * plan.shapes[m].first), (cuuint32_t)plan.shapes[m].second, 1};
        cuuint32_t es[3] = {1, 1, 1};
        if (enc_fn(&maps.m[m], CU_TENSOR_MAP_DATA_TYPE_FLOAT32, 3, enc_dev, dims, strides, box, es,
                   CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_NONE, CU_TENSOR_MAP_L2_PROMOTION_L2_128B,
                   CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE) != CUDA_SUCCESS)
            return KBMOD_ERR_UNSUPPORTED;
    }

    StagedParams prm;
    prm.psiphi = psiphi;
    prm.enc = reinterpret_cast<const u64*>(enc_dev);
    prm.plan = static_cast<const int*>(plan_dev);
    prm.vel = vel_dev;
    prm.status = status_dev;
    prm.nent = plan.nent; prm.N = N; prm.H = H; prm.W = W; prm.Wp = Wp; prm.K = K; prm.min_obs = min_obs;
    prm.y_begin = y_begin; prm.y_end = y_end;
    prm.tiles_x = (W + TW - 1) / TW;
    prm.tiles_y = (y_end - y_begin + TH - 1) / TH;
    prm.group_w = 8;
    const long long tiles = (long long)prm.tiles_x * prm.tiles_y;
    if (tiles > 0x7FFFFFFFLL) return KBMOD_ERR_UNSUPPORTED;
    if (tiles == 0) return KBMOD_OK;
    prm.ntiles = (int)tiles;
    prm.out = out;
    prm.dt = dt;
    int dev = 0, sms = 148;
    cudaGetDevice(&dev);
    cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev);
    const int grid = (int)std::min<long long>(tiles, sms);
    const int cm = N <= 16 ? 2 : (N <= 32 ? 1 : 0);
    if (K <= 8) {
        if (cm == 2) return launch_geom<2, 8>(geom, prm, maps, grid, st);
        if (cm == 1) return launch_geom<1, 8>(geom, prm, maps, grid, st);
        return launch_geom<0, 8>(geom, prm, maps, grid, st);
    }
    if (cm == 2) return launch_geom<2, 0>(geom, prm, maps, grid, st);
    if (cm == 1) return launch_geom<1, 0>(geom, prm, maps, grid, st);
    return launch_geom<0, 0>(geom, prm, maps, grid, st);
}

int launch_search_staged(const float2* psiphi, const DtTable& dt, int N, int H, int W,
                         const float* vel_host, int V, int K, int min_obs, int y_begin, int y_end,
                         const kbmod_result& out, void* plan_dev, const float2* vel_dev, float2* enc_dev,
                         int* status_dev, int geom, cudaStream_t st) {
    StagedPlan plan;
    if (int rc = staged_plan_build(dt, N, H, W, vel_host, V, geom, plan)) return rc;
    return staged_launch(plan, psiphi, dt, N, H, W, K, min_obs, y_begin, y_end, out, plan_dev, vel_dev, enc_dev,
                         status_dev, st);
}
}  // namespace kbmod
