// search_tiled.cu -- S3..S6, the fast path of kbmod_search (Eq.24-27).
//
// What makes it fast (and what it keeps exact):
//   * S3 is hoisted to the host.  d = fl(v*dt_i) is uniform over start pixels, and
//     ix = floor(fl(fl(x0+d)+0.5f)) equals x0 + floor(d+0.5) for EVERY integer x0 of the image
//     whenever frac(d) is farther from 0.5 than the two roundings can move the sum (a margin of a
//     few ulp of the largest coordinate).  The host proves that per (velocity, image) and stores
//     the integer shift; pairs it cannot prove ("unsafe") take the literal per-lane expression on
//     the device.  The sampled pixels are therefore identical to the definition, bit for bit.
//   * A CTA owns a tile of start pixels and walks the velocity grid in blocks of B neighbouring
//     velocities (host-ordered along a Hilbert curve in (vx,vy), so the B windows of an image
//     overlap and successive blocks touch neighbouring memory).  For a proven shift the 32 lanes of a
//     warp read 32 consecutive float2 samples at  base + offset[j][i]: one IMAD.WIDE + LDG.64 per
//     sample, no per-lane position arithmetic and no bounds test (the host-side bounding box of a
//     velocity's shifts decides once per (tile, velocity) whether every window is inside).
//   * The stack is re-encoded once per call (search_common.cuh) as (psi, -phi) with invalid samples = (+0,+0): one
//     packed add.rn.f32x2 accumulates both sums (adding +0 / -0 is exact, so the result equals the
//     in-order fp32 sum over valid observations), and the sign bit of the second word is the
//     validity flag, counted with one LEA.HI.  3 instructions per sample.
//   * Image 0 has dt = 0: its sample is the same for every velocity and is kept in registers.
//   * Per-pixel top-K lives in shared memory ((nu, vel_idx) x K per pixel, lane-interleaved so it
//     is bank-conflict free); the current K-th best is cached in registers and an approximate
//     Psi*rsqrt(Phi) pre-test keeps the correctly rounded div/sqrt and the list update off the
//     common path.  Psi/Phi/n_obs of the K winners are re-evaluated once at the end.
#include <algorithm>
#include <cmath>
#include <cstdlib>
#include <cstring>
#include <vector>

#include "search_common.cuh"
#include "search_tiled.cuh"
#include "topk_list.h"

namespace kbmod {

namespace {

constexpr int THREADS = 512;
constexpr int SH_SKIP = 0x7FFF7FFF;       // window outside any supported image
constexpr int SH_UNSAFE = (int)0x80008000;  // shift not proven: literal per-lane S3
constexpr int SH_LIMIT = 32000;
constexpr int META = 8;                   // ints of per-velocity meta data in a block record
//   meta[0] = original velocity index (or -1: padding)
//   meta[1] = sxlo | sxhi << 16   (int16 each)      bounding box of the proven shifts, images >= 1
//   meta[2] = sylo | syhi << 16
//   meta[3] = 1 if every image >= 1 has a proven, in-range shift
//   meta[4], meta[5] = vx, vy (float bits)

// record of one velocity block: off[B][N], sh[B][N], meta[B][META]
__host__ __device__ inline size_t rec_ints(int B, int N) { return (size_t)B * N * 2 + (size_t)B * META; }

int block_size_for_k(int K) { return K <= 8 ? 8 : (K <= 16 ? 16 : 32); }

}  // namespace

size_t tiled_plan_bytes(int N, int V, int K) {
    const int B = block_size_for_k(K);
    const size_t nblk = 2 * (((size_t)V + B - 1) / B);   // kernel 4 may split a block in two (see build_plan)
    return nblk * rec_ints(B, N) * sizeof(int) + 256;
}

static int build_plan(const DtTable& dt, int N, int H, int W, const float* vel, int V, int B,
                      std::vector<int>& plan, bool isolate);

int tiled_plan_build(const DtTable& dt, int N, int H, int W, const float* vel_host, int V, int K, bool queued,
                     TiledPlan& plan) {
    // limits of the int16 shift encoding and of the int32 element offsets
    if (W > 30000 || H > 30000) return KBMOD_ERR_UNSUPPORTED;
    if (queued && V >= (1 << 24)) return KBMOD_ERR_UNSUPPORTED;    // 25-bit velocity index in the queue word
    if ((long long)(N + 1) * H * enc_pitch(W) + (long long)SH_LIMIT * (enc_pitch(W) + 1) >= 0x7FFFFFFFLL) return KBMOD_ERR_UNSUPPORTED;
    plan.queued = queued;
    plan.nblk = build_plan(dt, N, H, W, vel_host, V, block_size_for_k(K), plan.rec, queued);
    if (plan.rec.size() * sizeof(int) > tiled_plan_bytes(N, V, K)) return KBMOD_ERR_UNSUPPORTED;
    return KBMOD_OK;
}

// Builds the host plan; returns the number of velocity blocks.  margin: see the header comment.
// isolate (kernel 4): a chunk of B velocities that contains velocities with an unproven or skipped
// shift is split into a block of the clean ones and a block of the others, and blocks are filled
// up with "benign" padding (never scored, proven shift (0,0): it samples the thread's own pixel),
// so that the clean block keeps the branch-free gather loops.  The per-pixel result does not
// depend on the order in which velocities are visited.
static int build_plan(const DtTable& dt, int N, int H, int W, const float* vel, int V, int B,
                      std::vector<int>& plan, bool isolate) {
    const std::vector<std::pair<unsigned, int>> key = hilbert_order(vel, V);    // processing order
    const int Wp = enc_pitch(W);        // row pitch of the encoded stack the element offsets refer to

    // largest coordinate magnitude any fl(x0 + d) can reach for an in-range window
    const double cmax = 2.0 * std::max(W, H) + 4.0;
    const double ulp = std::ldexp(1.0, (int)std::floor(std::log2(cmax)) - 23);
    const double margin = 4.0 * ulp;   // the two roundings move the sum by at most 1 ulp(cmax)

    // members of every block: a velocity index, PAD_SKIP (never scored, never sampled) or PAD_BENIGN
    constexpr int PAD_SKIP = -1, PAD_BENIGN = -2;
    std::vector<int> members;
    {
        auto dirty = [&](int j) {                // some image >= 1 has no proven in-range shift
            for (int i = 1; i < N; ++i) {
                volatile float dxf = vel[2 * j] * dt.dt[i];
                volatile float dyf = vel[2 * j + 1] * dt.dt[i];
                const double dx = dxf, dy = dyf;
                if (!(std::fabs(dx) < SH_LIMIT && std::fabs(dy) < SH_LIMIT)) return true;
                const double fx = dx - std::floor(dx), fy = dy - std::floor(dy);
                if (std::fabs(fx - 0.5) <= margin || std::fabs(fy - 0.5) <= margin) return true;
            }
            return false;
        };
        for (int c0 = 0; c0 < V; c0 += B) {
            const int c1 = std::min(V, c0 + B);
            std::vector<int> a, d;
            for (int jj = c0; jj < c1; ++jj) {
                const int j = key[jj].second;
                ((isolate && dirty(j)) ? d : a).push_back(j);
            }
            if (!a.empty()) {
                a.resize(B, isolate ? PAD_BENIGN : PAD_SKIP);
                members.insert(members.end(), a.begin(), a.end());
            }
            if (!d.empty()) {
                d.resize(B, PAD_SKIP);
                members.insert(members.end(), d.begin(), d.end());
            }
        }
    }
    const int nblk = (int)(members.size() / B);
    plan.assign((size_t)nblk * rec_ints(B, N), 0);
    for (int blk = 0; blk < nblk; ++blk) {
        int* off = plan.data() + (size_t)blk * rec_ints(B, N);
        int* sh = off + (size_t)B * N;
        int* meta = sh + (size_t)B * N;
        for (int b = 0; b < B; ++b) {
            const int j = members[(size_t)blk * B + b];
            int* m = meta + b * META;
            if (j == PAD_SKIP) {                 // padding velocity: never scored, never sampled
                m[0] = -1; m[3] = 0;
                for (int i = 0; i < N; ++i) { off[b * N + i] = 0; sh[b * N + i] = SH_SKIP; }
                continue;
            }
            if (j == PAD_BENIGN) {               // never scored; samples the thread's own pixel of image i
                m[0] = -1; m[1] = 0; m[2] = 0; m[3] = 1;
                for (int i = 0; i < N; ++i) {
                    off[b * N + i] = (int)((long long)i * H * Wp);
                    sh[b * N + i] = 0;           // proven shift (0, 0)
                }
                continue;
            }
            const float vx = vel[2 * j], vy = vel[2 * j + 1];
            m[0] = j;
            std::memcpy(&m[4], &vx, 4);
            std::memcpy(&m[5], &vy, 4);
            int sxlo = SH_LIMIT, sxhi = -SH_LIMIT, sylo = SH_LIMIT, syhi = -SH_LIMIT, all_ok = 1;
            for (int i = 0; i < N; ++i) {
                // d exactly as the device would form it: one fp32 multiply (never contracted)
                volatile float dxf = vx * dt.dt[i];
                volatile float dyf = vy * dt.dt[i];
                const double dx = dxf, dy = dyf;
                int code;
                long long o = 0;
                if (!(std::fabs(dx) < SH_LIMIT && std::fabs(dy) < SH_LIMIT)) {
                    code = SH_SKIP;              // farther than any supported image: no observation
                } else {
                    const double fx = dx - std::floor(dx), fy = dy - std::floor(dy);
                    if (std::fabs(fx - 0.5) <= margin || std::fabs(fy - 0.5) <= margin) {
                        code = SH_UNSAFE;
                    } else {
                        const int sx = (int)std::floor(dx + 0.5), sy = (int)std::floor(dy + 0.5);
                        code = (int)(((unsigned)sy << 16) | ((unsigned)sx & 0xFFFFu));
                        o = (long long)i * H * Wp + (long long)sy * Wp + sx;
                        if (i >= 1) {
                            sxlo = std::min(sxlo, sx); sxhi = std::max(sxhi, sx);
                            sylo = std::min(sylo, sy); syhi = std::max(syhi, sy);
                        }
                    }
                }
                if (i >= 1 && (code == SH_SKIP || code == SH_UNSAFE)) all_ok = 0;
                off[b * N + i] = (int)o;
                sh[b * N + i] = code;
            }
            if (N == 1) { sxlo = sxhi = sylo = syhi = 0; }
            m[1] = (int)(((unsigned)sxhi << 16) | ((unsigned)sxlo & 0xFFFFu));
            m[2] = (int)(((unsigned)syhi << 16) | ((unsigned)sylo & 0xFFFFu));
            m[3] = all_ok;
        }
    }
    return nblk;
}

// ---------------------------------------------------------------------------------------------
// device side
// ---------------------------------------------------------------------------------------------

typedef unsigned long long u64;

__device__ __forceinline__ void acc_add(u64& a, u64 s) {      // (Psi, -Phi) += (psi, -phi), RN each
#if defined(KBMOD_SIMT_EMUL)      // host build of the SIMT-emulation tests: two plain binary32 adds
    const float x = __fadd_rn(__uint_as_float((unsigned)a), __uint_as_float((unsigned)s));
    const float y = __fadd_rn(__uint_as_float((unsigned)(a >> 32)), __uint_as_float((unsigned)(s >> 32)));
    a = (u64)__float_as_uint(x) | ((u64)__float_as_uint(y) << 32);
#else
    asm("add.rn.f32x2 %0, %0, %1;" : "+l"(a) : "l"(s));
#endif
}
__device__ __forceinline__ u64 ld_sample(const u64* p) { return __ldg(p); }

struct TiledParams {
    const float2* psiphi;     // original stack (final re-evaluation of the winners)
    const u64* enc;           // encoded stack
    const int* plan;          // nblk records
    const float2* vel;        // caller's velocity table (device copy)
    int nblk, N, H, W, K, min_obs;
    int Wp;                   // row pitch of the encoded stack (W rounded up to even)
    int y_begin, y_end;       // band of start rows; the result planes hold rows y_begin..y_end-1 only
    int tiles_x, tiles_y, group_w;
    kbmod_result out;
    DtTable dt;
    // threshold mode (kbmod_search_threshold): every eligible trajectory with nu >= nu_min is appended
    kbmod_candidates cand;
    unsigned long long capacity;
    unsigned long long* count;
    float nu_min;
};

// RX x RY pixels per thread: x = tile_x + (warp % WX) * 32 * RX + rx * 32 + lane,
//                            y = tile_y + (warp / WX) * RY + ry
template <int RX, int RY, int WX, int B, int KMAX>
struct TileGeom {
    static constexpr int R = RX * RY;
    static constexpr int WARPS = THREADS / 32;
    static constexpr int TW = 32 * RX * WX;
    static constexpr int TH = RY * (WARPS / WX);
    static constexpr int PX = THREADS * R;
    static size_t smem_bytes(int N) {
        return (size_t)PX * KMAX * 8 + rec_ints(B, N) * sizeof(int);
    }
};

template <int RX, int RY, int WX, int B, int KMAX>
__global__ void __launch_bounds__(THREADS, 1)
search_tiled_kernel(const __grid_constant__ TiledParams prm) {
    using G = TileGeom<RX, RY, WX, B, KMAX>;
    constexpr int R = G::R;
    constexpr int PX = G::PX;
    extern __shared__ __align__(16) unsigned char smem_raw[];
    float* l_nu = reinterpret_cast<float*>(smem_raw);            // [KMAX][PX]
    int* l_idx = reinterpret_cast<int*>(l_nu + (size_t)KMAX * PX);   // [KMAX][PX]
    int* rec = l_idx + (size_t)KMAX * PX;                         // off[B][N], sh[B][N], meta[B][META]

    const int N = prm.N, H = prm.H, W = prm.W, K = prm.K;
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;

    // tile of this CTA: groups of group_w tile columns, row-major inside a group, so that the CTAs
    // running at the same time cover a compact region (their windows then share L2 lines)
    int tx, ty;
    {
        const int per_group = prm.group_w * prm.tiles_y;
        const int g = blockIdx.x / per_group, rem = blockIdx.x - g * per_group;
        const int gw = min(prm.group_w, prm.tiles_x - g * prm.group_w);
        ty = rem / gw;
        tx = g * prm.group_w + (rem - ty * gw);
    }
    const int tile_x = tx * G::TW, tile_y = prm.y_begin + ty * G::TH;
    const int x_first = tile_x + (warp % WX) * 32 * RX + lane;
    const int y_first = tile_y + (warp / WX) * RY;
    const int y_end = prm.y_end;                     // start rows of this search: [y_begin, y_end)
    const bool ragged = (tile_x + G::TW > W) || (tile_y + G::TH > y_end);
    // tile extent that holds real pixels (for window classification)
    const int tile_x1 = min(tile_x + G::TW, W) - 1, tile_y1 = min(tile_y + G::TH, y_end) - 1;

    const u64* basep[RY];
#pragma unroll
    for (int ry = 0; ry < RY; ++ry)
        basep[ry] = prm.enc + (size_t)min(y_first + ry, H - 1) * prm.Wp + min(x_first, W - 1);

    // per-pixel list state: nu of the worst entry (the K-th best once the list is full)
    float w_nu[R];
#pragma unroll
    for (int r = 0; r < R; ++r) {
        w_nu[r] = -INFINITY;
        for (int e = 0; e < K; ++e) {
            l_nu[e * PX + r * THREADS + tid] = -INFINITY;
            l_idx[e * PX + r * THREADS + tid] = 0x7FFFFFFF;
        }
    }

    const int rec_n = (int)rec_ints(B, N);
    int* r_off = rec;
    int* r_sh = rec + B * N;
    int* r_meta = rec + 2 * B * N;

    for (int blk = 0; blk < prm.nblk; ++blk) {
        __syncthreads();
        {
            const int* src = prm.plan + (size_t)blk * rec_n;
            for (int k = tid; k < rec_n; k += THREADS) rec[k] = __ldg(src + k);
        }
        __syncthreads();

        u64 acc[B][R];
        unsigned cnt[B][R];
        unsigned fast = 0;          // bit b: every window of velocity b is inside the image
#pragma unroll
        for (int b = 0; b < B; ++b) {
#pragma unroll
            for (int ry = 0; ry < RY; ++ry)
#pragma unroll
                for (int rx = 0; rx < RX; ++rx) {
                    // image 0 has dt = 0: shift (0,0) for every velocity
                    const bool inimg = (x_first + 32 * rx < W) && (y_first + ry < y_end);
                    const u64 s0 = inimg ? ld_sample(basep[ry] + 32 * rx) : 0ull;
                    acc[b][ry * RX + rx] = s0;
                    cnt[b][ry * RX + rx] = (unsigned)(s0 >> 63);
                }
            const int bx = r_meta[b * META + 1], by = r_meta[b * META + 2];
            const int sxlo = (short)(bx & 0xFFFF), sxhi = bx >> 16;
            const int sylo = (short)(by & 0xFFFF), syhi = by >> 16;
            const bool ok = r_meta[b * META + 3] && !ragged && tile_x + sxlo >= 0 &&
                            tile_x1 + sxhi < W && tile_y + sylo >= 0 && tile_y1 + syhi < H;
            fast |= ok ? (1u << b) : 0u;
        }

        for (int i = 1; i < N; ++i) {
#pragma unroll
            for (int b = 0; b < B; ++b) {
                if (fast & (1u << b)) {
                    const int o = r_off[b * N + i];
#pragma unroll
                    for (int ry = 0; ry < RY; ++ry) {
                        const u64* p = basep[ry] + o;
#pragma unroll
                        for (int rx = 0; rx < RX; ++rx) {
                            const u64 s = ld_sample(p + 32 * rx);
                            acc_add(acc[b][ry * RX + rx], s);
                            cnt[b][ry * RX + rx] += (unsigned)(s >> 63);
                        }
                    }
                } else {
                    const int code = r_sh[b * N + i];
                    if (code == SH_SKIP) continue;
                    const u64* img = prm.enc + (size_t)i * H * prm.Wp;
                    if (code != SH_UNSAFE) {
                        const int sx = (short)(code & 0xFFFF), sy = code >> 16;
                        // whole window outside: nothing to add (uniform over the CTA)
                        if (tile_x1 + sx < 0 || tile_x + sx >= W || tile_y1 + sy < 0 || tile_y + sy >= H)
                            continue;
#pragma unroll
                        for (int ry = 0; ry < RY; ++ry) {
                            const int y = y_first + ry + sy;
                            const bool yin = (y_first + ry < y_end) && y >= 0 && y < H;
#pragma unroll
                            for (int rx = 0; rx < RX; ++rx) {
                                const int x = x_first + 32 * rx + sx;
                                const bool in = yin && (x_first + 32 * rx < W) && x >= 0 && x < W;
                                const u64 s = in ? ld_sample(img + (size_t)y * prm.Wp + x) : 0ull;
                                acc_add(acc[b][ry * RX + rx], s);
                                cnt[b][ry * RX + rx] += (unsigned)(s >> 63);
                            }
                        }
                    } else {
                        const float vx = __int_as_float(r_meta[b * META + 4]);
                        const float vy = __int_as_float(r_meta[b * META + 5]);
                        const float dti = prm.dt.dt[i];
#pragma unroll
                        for (int ry = 0; ry < RY; ++ry) {
                            int y = 0;
                            const bool yin = traj_pixel(y_first + ry, vy, dti, H, y) && (y_first + ry < y_end);
#pragma unroll
                            for (int rx = 0; rx < RX; ++rx) {
                                int x = 0;
                                const bool in = traj_pixel(x_first + 32 * rx, vx, dti, W, x) && yin &&
                                                (x_first + 32 * rx < W);
                                const u64 s = in ? ld_sample(img + (size_t)y * prm.Wp + x) : 0ull;
                                acc_add(acc[b][ry * RX + rx], s);
                                cnt[b][ry * RX + rx] += (unsigned)(s >> 63);
                            }
                        }
                    }
                }
            }
        }

        // S5 + S6 for the B x R trajectories of this block
#pragma unroll
        for (int b = 0; b < B; ++b) {
            const int j = r_meta[b * META + 0];
            if (j < 0) continue;
#pragma unroll
            for (int r = 0; r < R; ++r) {
                const float Psi = __uint_as_float((unsigned)acc[b][r]);
                const float Phi = 0.0f - __uint_as_float((unsigned)(acc[b][r] >> 32));
                if ((int)cnt[b][r] >= prm.min_obs && Phi > 0.0f) {
                    const float approx = Psi * rsqrtf(Phi);
                    const float lo = fmaf(-fabsf(w_nu[r]), 4e-6f, w_nu[r]);   // -inf stays -inf
                    if (!(approx < lo)) {
                        const float nu = score_nu(Psi, Phi);
                        const int p = r * THREADS + tid;
                        // worst (smallest nu, ties -> larger index) and second-worst entries
                        float wn = INFINITY, vn = INFINITY;
                        int wj = -1, vj = -1, ws = 0;
                        for (int e = 0; e < K; ++e) {
                            const float ne = l_nu[e * PX + p];
                            const int je = l_idx[e * PX + p];
                            if (ne < wn || (ne == wn && je > wj)) {
                                vn = wn; vj = wj;
                                wn = ne; wj = je; ws = e;
                            } else if (ne < vn || (ne == vn && je > vj)) {
                                vn = ne; vj = je;
                            }
                        }
                        if (nu > wn || (nu == wn && j < wj)) {
                            l_nu[ws * PX + p] = nu;
                            l_idx[ws * PX + p] = j;
                            // the new worst is the old second-worst or the candidate itself
                            w_nu[r] = (nu < vn || (nu == vn && j > vj)) ? nu : vn;
                        }
                    }
                }
            }
        }
    }

    // ---- output: K entries per pixel, best first; winners re-evaluated with the literal S3+S4
#pragma unroll 1
    for (int r = 0; r < R; ++r) {
        const int rx = r % RX, ry = r / RX;
        const int x0 = x_first + 32 * rx, y0 = y_first + ry;
        if (x0 >= W || y0 >= y_end) continue;
        const int p = r * THREADS + tid;
        const size_t obase = ((size_t)(y0 - prm.y_begin) * W + x0) * K;
        for (int k = 0; k < K; ++k) {
            float bn = -INFINITY;
            int bj = 0x7FFFFFFF, bs = -1;
            for (int e = 0; e < K; ++e) {
                const float ne = l_nu[e * PX + p];
                const int je = l_idx[e * PX + p];
                if (je != 0x7FFFFFFF && (bs < 0 || ne > bn || (ne == bn && je < bj))) { bn = ne; bj = je; bs = e; }
            }
            if (bs >= 0) {
                l_idx[bs * PX + p] = 0x7FFFFFFF;
                // literal evaluation (bit-identical sums: same samples, same order)
                float Psi = 0.0f, Phi = 0.0f;
                int n = 0;
                const float2 v = __ldg(prm.vel + bj);
                for (int i = 0; i < N; ++i) {
                    int ix, iy;
                    if (traj_pixel(x0, v.x, prm.dt.dt[i], W, ix) && traj_pixel(y0, v.y, prm.dt.dt[i], H, iy)) {
                        const float2 s = __ldg(prm.psiphi + ((size_t)i * H + iy) * W + ix);
                        if (s.x == s.x) { Psi = __fadd_rn(Psi, s.x); Phi = __fadd_rn(Phi, s.y); ++n; }
                    }
                }
                prm.out.vel_idx[obase + k] = bj;
                prm.out.n_obs[obase + k] = n;
                prm.out.psi[obase + k] = Psi;
                prm.out.phi[obase + k] = Phi;
                prm.out.nu[obase + k] = score_nu(Psi, Phi);
                prm.out.alpha[obase + k] = score_alpha(Psi, Phi);
            } else {
                prm.out.vel_idx[obase + k] = -1;
                prm.out.n_obs[obase + k] = 0;
                prm.out.psi[obase + k] = 0.0f;
                prm.out.phi[obase + k] = 0.0f;
                prm.out.nu[obase + k] = -INFINITY;
                prm.out.alpha[obase + k] = 0.0f;
            }
        }
    }
}

// ---------------------------------------------------------------------------------------------
// Kernel 4: the same gathers, S5/S6 off the common path (queue-compacted top-K)
// ---------------------------------------------------------------------------------------------
// search_tiled_kernel spends three quarters of its instructions in the shared-memory list code,
// because a warp enters it whenever ANY of its 32 lanes passes the pre-test (ncu, profiles/
// r01_v2_tiled.md).  Here the survivors of the pre-test are compacted by ballot into a per-warp
// shared-memory queue and handled 32 at a time, one lane per candidate: correctly rounded
// score, sorted insert into the pixel's list.  The lists live in the nu / vel_idx output planes
// (only the owning warp touches a pixel's list, through L2), so shared memory holds only the
// block record and the queues.  S5/S6 are the code of the staged kernel (search_staged.cu),
// whose logic tests/test_staged_simt.py checks on the CPU; S3/S4 are search_tiled_kernel's.
constexpr int QCAP = 64;                  // per-warp candidate queue entries (power of two, >= 63)

struct ListMemPlanes {                    // list entries are read and written through L2
    template <class T> static __device__ __forceinline__ T ld(const T* p) { return __ldcg(p); }
    template <class T> static __device__ __forceinline__ void st(T* p, T v) { __stcg(p, v); }
};

// One dense pass over up to 32 queued candidates of this warp: lane l takes entry qhead + l.
// THRESH: the candidate is appended to the compacted list if its exactly scored nu >= nu_min.
template <int RX, int KP, bool THRESH>
__device__ __forceinline__ void process_batch_q(const TiledParams& prm, const float* q_psi, const float* q_phi,
                                                const unsigned* q_meta, unsigned qhead, int n, int lane,
                                                int wx0, int wy0) {
    bool valid = lane < n;
    const unsigned idx = (qhead + lane) & (QCAP - 1);
    const float Psi = q_psi[idx], Phi = q_phi[idx];
    const unsigned meta = q_meta[idx];
    const int pix = meta & 127, j = (int)(meta >> 7);
    const int r = pix >> 5, ln = pix & 31;
    const int x = wx0 + ln + 32 * (r % RX), y = wy0 + r / RX;
    const float nu = valid ? score_nu(Psi, Phi) : 0.0f;
    if constexpr (THRESH) {
        if (valid && nu >= prm.nu_min) {
            // the sums in the queue are the in-order fp32 sums already; the literal walk adds n_obs
            float lPsi = 0.0f, lPhi = 0.0f;
            int cnt = 0;
            const float2 v = __ldg(prm.vel + j);
            for (int i = 0; i < prm.N; ++i) {
                int ix, iy;
                if (traj_pixel(x, v.x, prm.dt.dt[i], prm.W, ix) && traj_pixel(y, v.y, prm.dt.dt[i], prm.H, iy)) {
                    const float2 s = __ldg(prm.psiphi + ((size_t)i * prm.H + iy) * prm.W + ix);
                    if (s.x == s.x) { lPsi = __fadd_rn(lPsi, s.x); lPhi = __fadd_rn(lPhi, s.y); ++cnt; }
                }
            }
            const unsigned long long slot = atomicAdd(prm.count, 1ull);
            if (slot < prm.capacity) {
                prm.cand.x[slot] = x; prm.cand.y[slot] = y; prm.cand.vel_idx[slot] = j; prm.cand.n_obs[slot] = cnt;
                prm.cand.psi[slot] = lPsi; prm.cand.phi[slot] = lPhi; prm.cand.nu[slot] = score_nu(lPsi, lPhi);
                prm.cand.alpha[slot] = score_alpha(lPsi, lPhi);
            }
        }
        return;
    }
    const size_t p = valid ? ((size_t)(y - prm.y_begin) * prm.W + x) * prm.K : 0;
    for (;;) {
        // two candidates of the same pixel in one batch: lowest lane first, the rest next round
        const unsigned same = __match_any_sync(0xFFFFFFFFu, valid ? pix : 128 + lane);
        if (valid && lane == __ffs(same) - 1) {
            list_insert<KP, ListMemPlanes>(prm.out.nu + p, prm.out.vel_idx + p, prm.K, nu, j);
            valid = false;
        }
        __syncwarp();
        if (!__any_sync(0xFFFFFFFFu, valid)) break;
    }
}

// RX x RY pixels per thread: x = tile_x + rx * 32 + lane, y = tile_y + warp * RY + ry; B * RX * RY = 32.
// CM: how valid samples are counted.  0: one additive counter per (velocity, pixel).  2 (RX = 2,
// N <= 16): the sign bits are shifted into a history word shared by the two rx pixels of a row
// (rx = 0 lands on the odd bits, rx = 1 on the even ones) and counted with popc when the block is
// scored: half the counter registers, so more gathers can be in flight.
template <int RX, int RY, int B, int KP, int CM, bool THRESH = false>
__global__ void __launch_bounds__(THREADS, 1)
search_tiledq_kernel(const __grid_constant__ TiledParams prm) {
    constexpr int R = RX * RY;
    static_assert(B * R == 32, "the scoring switch lists B*R = 32 steps");
    static_assert(CM == 0 || (CM == 2 && RX == 2), "history counting pairs the two rx pixels of a row");
    constexpr int NC = (CM == 2) ? RY : R;        // count registers per velocity
    constexpr int TW = 32 * RX, TH = RY * (THREADS / 32);
    extern __shared__ __align__(16) unsigned char smem_raw[];
    const int N = prm.N, H = prm.H, W = prm.W, K = prm.K;
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const int rec_n = (int)rec_ints(B, N);
    int* rec2 = reinterpret_cast<int*>(smem_raw);                 // two block records (double buffer)
    float* q_psi = reinterpret_cast<float*>(rec2 + 2 * rec_n) + warp * (3 * QCAP);
    float* q_phi = q_psi + QCAP;
    unsigned* q_meta = reinterpret_cast<unsigned*>(q_phi + QCAP);

    int tx, ty;                                                   // tile order: see search_tiled_kernel
    {
        const int per_group = prm.group_w * prm.tiles_y;
        const int g = blockIdx.x / per_group, rem = blockIdx.x - g * per_group;
        const int gw = min(prm.group_w, prm.tiles_x - g * prm.group_w);
        ty = rem / gw;
        tx = g * prm.group_w + (rem - ty * gw);
    }
    const int tile_x = tx * TW, tile_y = prm.y_begin + ty * TH;
    const int x_first = tile_x + lane;
    const int y_first = tile_y + warp * RY;
    const int y_end = prm.y_end;                                  // start rows of this search: [y_begin, y_end)
    const bool ragged = (tile_x + TW > W) || (tile_y + TH > y_end);
    const int tile_x1 = min(tile_x + TW, W) - 1, tile_y1 = min(tile_y + TH, y_end) - 1;
    unsigned inimg = 0;                                           // bit r: pixel r of this thread is a start pixel of the band
#pragma unroll
    for (int r = 0; r < R; ++r)
        inimg |= ((x_first + 32 * (r % RX) < W) && (y_first + r / RX < y_end)) ? (1u << r) : 0u;
    // result-plane position (band-relative rows) of pixel r: pix0 + 32*rx + ry*W
    const size_t pix0 = (size_t)(y_first - prm.y_begin) * W + x_first;

    const u64* basep[RY];
#pragma unroll
    for (int ry = 0; ry < RY; ++ry)
        basep[ry] = prm.enc + (size_t)min(y_first + ry, H - 1) * prm.Wp + min(x_first, W - 1);

#if !defined(KBMOD_SIMT_EMUL)
    // keep the row pointers as opaque 64-bit registers: `basep[ry] + o` is then one IMAD.WIDE per
    // pair of gathers instead of a 64-bit index add plus a 64-bit scale-and-add (4 instructions)
#pragma unroll
    for (int ry = 0; ry < RY; ++ry) asm volatile("" : "+l"(basep[ry]));
#endif

    // empty lists (in the output planes)
    if constexpr (!THRESH)
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
    const unsigned minobs = (unsigned)prm.min_obs;

    // block records are double-buffered: record blk+1 is fetched while block blk is computed, and
    // one barrier per block both publishes it and retires record blk
    for (int k = tid; k < rec_n; k += THREADS) rec2[k] = __ldg(prm.plan + k);
    __syncthreads();

    for (int blk = 0; blk < prm.nblk; ++blk) {
        const int* rec = rec2 + (blk & 1) * rec_n;                // off[B][N], sh[B][N], meta[B][META]
        const int* r_off = rec;
        const int* r_sh = rec + B * N;
        const int* r_meta = rec + 2 * B * N;
        if (blk + 1 < prm.nblk) {
            const int* src = prm.plan + (size_t)(blk + 1) * rec_n;
            int* dst = rec2 + ((blk + 1) & 1) * rec_n;
            for (int k = tid; k < rec_n; k += THREADS) dst[k] = __ldg(src + k);
        }

        float lo[R];                               // pre-test bound: K-th best nu minus a safety margin
#pragma unroll
        for (int r = 0; r < R; ++r) {
            float w = -INFINITY;
            if constexpr (THRESH) {
                w = prm.nu_min;                                  // fixed bound: the detection threshold
            } else {
                if (inimg & (1u << r))
                    w = __ldcg(prm.out.nu + (pix0 + 32 * (r % RX) + (size_t)(r / RX) * W) * K + (K - 1));
            }
            lo[r] = fmaf(-fabsf(w), 4e-6f, w);                   // -inf stays -inf
        }

        u64 acc[B][R];
        unsigned cnt[B][NC];
        unsigned fast = 0;          // bit b: every window of velocity b is inside the image
        bool proven = true;         // every (velocity, image >= 1) of the block has a proven integer shift
        // one sample of pixel r (= ry * RX + rx) of velocity b: the packed add and the validity count
        auto take = [&](int b, int r, u64 s) {
            acc_add(acc[b][r], s);
            if constexpr (CM == 2) cnt[b][r / RX] = __funnelshift_l((unsigned)(s >> 32), cnt[b][r / RX], 1);
            else cnt[b][r] += (unsigned)(s >> 63);
        };
#pragma unroll
        for (int b = 0; b < B; ++b) {
#pragma unroll
            for (int r = 0; r < R; ++r) {
                // image 0 has dt = 0: shift (0,0) for every velocity
                const u64 s0 = (inimg & (1u << r)) ? ld_sample(basep[r / RX] + 32 * (r % RX)) : 0ull;
                acc[b][r] = s0;
                if constexpr (CM == 2) cnt[b][r / RX] = (r % RX) ? cnt[b][r / RX] * 2u + (unsigned)(s0 >> 63) : (unsigned)(s0 >> 63);
                else cnt[b][r] = (unsigned)(s0 >> 63);
            }
            const int bx = r_meta[b * META + 1], by = r_meta[b * META + 2];
            const int sxlo = (short)(bx & 0xFFFF), sxhi = bx >> 16;
            const int sylo = (short)(by & 0xFFFF), syhi = by >> 16;
            const bool ok = r_meta[b * META + 3] && !ragged && tile_x + sxlo >= 0 &&
                            tile_x1 + sxhi < W && tile_y + sylo >= 0 && tile_y1 + syhi < H;
            fast |= ok ? (1u << b) : 0u;
            proven = proven && (r_meta[b * META + 3] != 0);
        }

        if (fast == (B == 32 ? 0xFFFFFFFFu : (1u << B) - 1u)) {
            // every window of every velocity of the block is inside the image (interior tiles):
            // straight-line code per image, so the B x R independent loads can be issued ahead of
            // the adds (the per-velocity branches of the general loop below keep only R in flight)
            for (int i = 1; i < N; ++i) {
#pragma unroll
                for (int b = 0; b < B; ++b) {
                    const int o = r_off[b * N + i];
#pragma unroll
                    for (int ry = 0; ry < RY; ++ry) {
                        const u64* p = basep[ry] + o;
#pragma unroll
                        for (int rx = 0; rx < RX; ++rx) {
                            const u64 s = ld_sample(p + 32 * rx);
                            take(b, ry * RX + rx, s);
                        }
                    }
                }
            }
        } else if (proven) {
            // every shift of the block is proven but some windows cross the image border (or the
            // tile is ragged): still straight-line code, each lane tests its own sample position
            for (int i = 1; i < N; ++i) {
#pragma unroll
                for (int b = 0; b < B; ++b) {
                    const int o = r_off[b * N + i];
                    const int code = r_sh[b * N + i];
                    const int sx = (short)(code & 0xFFFF), sy = code >> 16;
#pragma unroll
                    for (int ry = 0; ry < RY; ++ry) {
                        const bool yin = (unsigned)(y_first + ry + sy) < (unsigned)H;
                        const u64* p = basep[ry] + o;       // = enc + ((i*H + y)*W + x) for pixels inside the image
#pragma unroll
                        for (int rx = 0; rx < RX; ++rx) {
                            const bool in = yin && ((inimg >> (ry * RX + rx)) & 1u) &&
                                            (unsigned)(x_first + 32 * rx + sx) < (unsigned)W;
                            const u64 s = in ? ld_sample(p + 32 * rx) : 0ull;
                            take(b, ry * RX + rx, s);
                        }
                    }
                }
            }
        } else
        for (int i = 1; i < N; ++i) {
#pragma unroll
            for (int b = 0; b < B; ++b) {
                if (fast & (1u << b)) {
                    const int o = r_off[b * N + i];
#pragma unroll
                    for (int ry = 0; ry < RY; ++ry) {
                        const u64* p = basep[ry] + o;
#pragma unroll
                        for (int rx = 0; rx < RX; ++rx) {
                            const u64 s = ld_sample(p + 32 * rx);
                            take(b, ry * RX + rx, s);
                        }
                    }
                } else {
                    const int code = r_sh[b * N + i];
                    if (code == SH_SKIP) continue;
                    const u64* img = prm.enc + (size_t)i * H * prm.Wp;
                    if (code != SH_UNSAFE) {
                        const int sx = (short)(code & 0xFFFF), sy = code >> 16;
                        // whole window outside: nothing to add (uniform over the CTA)
                        if (tile_x1 + sx < 0 || tile_x + sx >= W || tile_y1 + sy < 0 || tile_y + sy >= H)
                            continue;
#pragma unroll
                        for (int ry = 0; ry < RY; ++ry) {
                            const int y = y_first + ry + sy;
                            const bool yin = (y_first + ry < y_end) && y >= 0 && y < H;
#pragma unroll
                            for (int rx = 0; rx < RX; ++rx) {
                                const int x = x_first + 32 * rx + sx;
                                const bool in = yin && (x_first + 32 * rx < W) && x >= 0 && x < W;
                                const u64 s = in ? ld_sample(img + (size_t)y * prm.Wp + x) : 0ull;
                                take(b, ry * RX + rx, s);
                            }
                        }
                    } else {
                        const float vx = __int_as_float(r_meta[b * META + 4]);
                        const float vy = __int_as_float(r_meta[b * META + 5]);
                        const float dti = prm.dt.dt[i];
#pragma unroll
                        for (int ry = 0; ry < RY; ++ry) {
                            int y = 0;
                            const bool yin = traj_pixel(y_first + ry, vy, dti, H, y) && (y_first + ry < y_end);
#pragma unroll
                            for (int rx = 0; rx < RX; ++rx) {
                                int x = 0;
                                const bool in = traj_pixel(x_first + 32 * rx, vx, dti, W, x) && yin &&
                                                (x_first + 32 * rx < W);
                                const u64 s = in ? ld_sample(img + (size_t)y * prm.Wp + x) : 0ull;
                                take(b, ry * RX + rx, s);
                            }
                        }
                    }
                }
            }
        }

        // ---- S5 + S6 for the B x R trajectories of this block.  The steps are the cases of one
        // switch so that a single copy of the batch code serves all of them: a step that fills the
        // queue to 32 leaves the switch, the batch is processed, and the switch is re-entered at
        // the next step.
        int step = 0;
        for (;;) {
            bool flush = false;
            switch (step) {
#define KBMOD_VEL_OF(b) r_meta[(b) * META + 0]
#define KBMOD_QPUT(qi, Psi, Phi, meta) (q_psi[qi] = (Psi), q_phi[qi] = (Phi), q_meta[qi] = (meta))
                KBMOD_SCORE_STEPS_32(KBMOD_VEL_OF, KBMOD_QPUT)
#undef KBMOD_VEL_OF
#undef KBMOD_QPUT
                default: break;
            }
            if (!flush) break;
            __syncwarp();
            process_batch_q<RX, KP, THRESH>(prm, q_psi, q_phi, q_meta, qhead, 32, lane, tile_x, y_first);
            qhead += 32;
        }
        __syncthreads();
    }

    // ---- end of tile: drain the queue, then re-evaluate the winners literally and write them
    __syncwarp();
    while (qtail != qhead) {
        const int n = (int)min(32u, qtail - qhead);
        process_batch_q<RX, KP, THRESH>(prm, q_psi, q_phi, q_meta, qhead, n, lane, tile_x, y_first);
        qhead += n;
    }
    __syncwarp();
    if constexpr (THRESH) return;                       // no per-pixel lists to finish
#pragma unroll 1
    for (int r = 0; r < R; ++r) {
        if (!(inimg & (1u << r))) continue;
        const int x0 = x_first + 32 * (r % RX), y0 = y_first + r / RX;
        const size_t obase = ((size_t)(y0 - prm.y_begin) * W + x0) * K;
        for (int k = 0; k < K; ++k) {
            const int bj = __ldcg(prm.out.vel_idx + obase + k);
            if (bj != LIST_EMPTY_IDX) {
                // literal evaluation (bit-identical sums: same samples, same order)
                float Psi = 0.0f, Phi = 0.0f;
                int n = 0;
                const float2 v = __ldg(prm.vel + bj);
                for (int i = 0; i < N; ++i) {
                    int ix, iy;
                    if (traj_pixel(x0, v.x, prm.dt.dt[i], W, ix) && traj_pixel(y0, v.y, prm.dt.dt[i], H, iy)) {
                        const float2 s = __ldg(prm.psiphi + ((size_t)i * H + iy) * W + ix);
                        if (s.x == s.x) { Psi = __fadd_rn(Psi, s.x); Phi = __fadd_rn(Phi, s.y); ++n; }
                    }
                }
                prm.out.n_obs[obase + k] = n;
                prm.out.psi[obase + k] = Psi;
                prm.out.phi[obase + k] = Phi;
                prm.out.nu[obase + k] = score_nu(Psi, Phi);
                prm.out.alpha[obase + k] = score_alpha(Psi, Phi);
            } else {
                prm.out.vel_idx[obase + k] = -1;
                prm.out.n_obs[obase + k] = 0;
                prm.out.psi[obase + k] = 0.0f;
                prm.out.phi[obase + k] = 0.0f;
                prm.out.nu[obase + k] = -INFINITY;
                prm.out.alpha[obase + k] = 0.0f;
            }
        }
    }
}

// ---------------------------------------------------------------------------------------------
// launch
// ---------------------------------------------------------------------------------------------
template <int RX, int RY, int WX, int B, int KMAX>
static int launch_variant(TiledParams& prm, int group_w, cudaStream_t st) {
    using G = TileGeom<RX, RY, WX, B, KMAX>;
    const size_t smem = G::smem_bytes(prm.N);
    if (smem > 227 * 1024) return KBMOD_ERR_UNSUPPORTED;
    auto kern = search_tiled_kernel<RX, RY, WX, B, KMAX>;
    // per launch, not cached: the attribute belongs to the current device's copy of the function
    if (cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, 227 * 1024) != cudaSuccess)
        return KBMOD_ERR_CUDA;
    prm.tiles_x = (prm.W + G::TW - 1) / G::TW;
    prm.tiles_y = (prm.y_end - prm.y_begin + G::TH - 1) / G::TH;
    prm.group_w = group_w > 0 ? std::min(group_w, 256) : std::max(1, 512 / G::TW);
    const long long tiles = (long long)prm.tiles_x * prm.tiles_y;
    if (tiles > 0x7FFFFFFFLL) return KBMOD_ERR_UNSUPPORTED;
    if (tiles == 0) return KBMOD_OK;
    KBMOD_LAUNCH(kern, (unsigned)tiles, THREADS, smem, st, prm);
    note_launch();
    return cudaGetLastError() == cudaSuccess ? KBMOD_OK : KBMOD_ERR_CUDA;
}

template <int RX, int RY, int B, int KP, int CM, bool THRESH = false>
static int launch_variant_q(TiledParams& prm, int group_w, cudaStream_t st) {
    constexpr int TW = 32 * RX, TH = RY * (THREADS / 32);
    // two block records + the queues: 14.7 KB at N = 15, 46.8 KB at most (N = 64, B = 32), i.e. below
    // the 48 KB that need no opt-in; the rest of the SM's 256 KB stays L1 for the gathers
    const size_t smem = 2 * rec_ints(B, prm.N) * sizeof(int) + (size_t)(THREADS / 32) * QCAP * 12;
    if (smem > 48 * 1024) return KBMOD_ERR_UNSUPPORTED;
    auto kern = search_tiledq_kernel<RX, RY, B, KP, CM, THRESH>;
    prm.tiles_x = (prm.W + TW - 1) / TW;
    prm.tiles_y = (prm.y_end - prm.y_begin + TH - 1) / TH;
    // tile rasterisation: groups of group_w tile columns (default 512 px wide; kbmod_search_options
    // tile_group_w overrides it: a tuning knob, the results do not depend on it)
    prm.group_w = group_w > 0 ? std::min(group_w, 256) : std::max(1, 512 / TW);
    const long long tiles = (long long)prm.tiles_x * prm.tiles_y;
    if (tiles > 0x7FFFFFFFLL) return KBMOD_ERR_UNSUPPORTED;
    if (tiles == 0) return KBMOD_OK;
    KBMOD_LAUNCH(kern, (unsigned)tiles, THREADS, smem, st, prm);
    note_launch();
    return cudaGetLastError() == cudaSuccess ? KBMOD_OK : KBMOD_ERR_CUDA;
}

int tiled_launch(const TiledPlan& plan, const float2* psiphi, const DtTable& dt, int N, int H, int W, int K,
                 int min_obs, int y_begin, int y_end, const kbmod_result& out, void* plan_dev,
                 const float2* vel_dev, float2* enc_dev, int group_w, cudaStream_t st) {
    if (cudaMemcpyAsync(plan_dev, plan.rec.data(), plan.rec.size() * sizeof(int), cudaMemcpyHostToDevice, st) != cudaSuccess)
        return KBMOD_ERR_CUDA;

    KBMOD_LAUNCH(encode_kernel, 148 * 8, 256, 0, st, psiphi, reinterpret_cast<float4*>(enc_dev), W, enc_pitch(W),
                 (size_t)N * H);
    note_launch();
    if (cudaGetLastError() != cudaSuccess) return KBMOD_ERR_CUDA;

    TiledParams prm;
    prm.psiphi = psiphi;
    prm.enc = reinterpret_cast<const u64*>(enc_dev);
    prm.plan = static_cast<const int*>(plan_dev);
    prm.vel = vel_dev;
    prm.nblk = plan.nblk; prm.N = N; prm.H = H; prm.W = W; prm.K = K; prm.min_obs = min_obs;
    prm.Wp = enc_pitch(W);
    prm.y_begin = y_begin; prm.y_end = y_end;
    prm.out = out;
    prm.dt = dt;
    std::memset(&prm.cand, 0, sizeof(prm.cand));
    prm.capacity = 0; prm.count = nullptr; prm.nu_min = 0.0f;
    if (plan.queued) {                                              // kernel 4: same tiles, queue-compacted S5/S6
        const bool hist = N <= 16;                                  // history-bit counting (see CM)
        if (K <= 8) return hist ? launch_variant_q<2, 2, 8, 8, 2>(prm, group_w, st) : launch_variant_q<2, 2, 8, 8, 0>(prm, group_w, st);
        if (K <= 16) return hist ? launch_variant_q<2, 1, 16, 0, 2>(prm, group_w, st) : launch_variant_q<2, 1, 16, 0, 0>(prm, group_w, st);
        return launch_variant_q<1, 1, 32, 0, 0>(prm, group_w, st);
    }
    if (K <= 8) return launch_variant<2, 2, 1, 8, 8>(prm, group_w, st);      // tile 64 x 32
    if (K <= 16) return launch_variant<2, 1, 1, 16, 16>(prm, group_w, st);   // tile 64 x 16
    return launch_variant<1, 1, 1, 32, 32>(prm, group_w, st);                // tile 32 x 16
}

int tiled_launch_threshold(const TiledPlan& plan, const float2* psiphi, const DtTable& dt, int N, int H, int W,
                           int min_obs, float nu_min, int y_begin, int y_end, const kbmod_candidates& cand,
                           unsigned long long capacity, unsigned long long* count, void* plan_dev,
                           const float2* vel_dev, float2* enc_dev, int group_w, cudaStream_t st) {
    if (!plan.queued) return KBMOD_ERR_ARG;
    if (cudaMemcpyAsync(plan_dev, plan.rec.data(), plan.rec.size() * sizeof(int), cudaMemcpyHostToDevice, st) != cudaSuccess)
        return KBMOD_ERR_CUDA;
    KBMOD_LAUNCH(encode_kernel, 148 * 8, 256, 0, st, psiphi, reinterpret_cast<float4*>(enc_dev), W, enc_pitch(W),
                 (size_t)N * H);
    note_launch();
    if (cudaGetLastError() != cudaSuccess) return KBMOD_ERR_CUDA;
    TiledParams prm;
    std::memset(&prm.out, 0, sizeof(prm.out));
    prm.psiphi = psiphi;
    prm.enc = reinterpret_cast<const u64*>(enc_dev);
    prm.plan = static_cast<const int*>(plan_dev);
    prm.vel = vel_dev;
    prm.nblk = plan.nblk; prm.N = N; prm.H = H; prm.W = W; prm.K = 8; prm.min_obs = min_obs;   // plan blocks of 8
    prm.Wp = enc_pitch(W);
    prm.y_begin = y_begin; prm.y_end = y_end;
    prm.dt = dt;
    prm.cand = cand; prm.capacity = capacity; prm.count = count; prm.nu_min = nu_min;
    return N <= 16 ? launch_variant_q<2, 2, 8, 8, 2, true>(prm, group_w, st)
                   : launch_variant_q<2, 2, 8, 8, 0, true>(prm, group_w, st);
}

int launch_search_tiled(const float2* psiphi, const DtTable& dt, int N, int H, int W,
                        const float* vel_host, int V, int K, int min_obs, int y_begin, int y_end,
                        const kbmod_result& out, void* plan_dev, const float2* vel_dev, float2* enc_dev,
                        bool queued, int group_w, cudaStream_t st) {
    TiledPlan plan;
    if (int rc = tiled_plan_build(dt, N, H, W, vel_host, V, K, queued, plan)) return rc;
    return tiled_launch(plan, psiphi, dt, N, H, W, K, min_obs, y_begin, y_end, out, plan_dev, vel_dev, enc_dev,
                        group_w, st);
}

}  // namespace kbmod
