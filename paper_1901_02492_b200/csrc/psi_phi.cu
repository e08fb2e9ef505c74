// psi_phi.cu -- S1+S2: likelihood images Psi_i, Phi_i (Eq.19-20).
//
//   Psi(y) = sum_d s(y+d) T(d),  Phi(y) = sum_d w(y+d) T(d)^2,   s = sci/var, w = 1/var on good
//   pixels and 0 elsewhere (masked, non-finite, var <= 0, outside the image: P:171).
//
// General 2-D single-pass kernel (arbitrary, non-separable T; "single pass ... to support
// non-Gaussian PSF's"): one CTA = one 64 x 32 output tile of one image.  The tile + halo of s and
// w is formed once (S1 fused, never stored to HBM) and kept in shared memory as two fp32 planes;
// each thread produces a strip of 8 outputs along x from a register window that slides over dx,
// so one LDS.128 feeds 8 FMAs.  T and T^2 sit in shared memory and are read as broadcast LDS.128.
// The 8 lanes of a quarter warp cover 4 strips x 2 rows with an odd row pitch (in 16-byte units),
// which makes every LDS.128 bank-conflict free.  Output is the interleaved float2 (psi, phi).
//
// Round 2 (BASELINE.json subsystem (1) "float4 coalesced I/O"):
//   * the whole stack in one launch (blockIdx.x = image * tiles + tile); the PSFs travel in one
//     32 KB kernel parameter, so a launch takes floor(8000 / P^2) images (18 at P = 21, 10 at
//     P = 27): config 3 is ONE launch instead of 15;
//   * the halo stage reads sci and var as float4 and the mask as 4-byte words from a 16-byte
//     aligned superset of the halo (W % 4 == 0 and aligned bases; otherwise the scalar stage);
//   * the outputs go through shared memory so that a warp stores 32 consecutive 16-byte vectors
//     (two pixels each) per instruction instead of 32 8-byte values 64 bytes apart.
// The arithmetic -- which products are formed, in which order they are added -- is unchanged, so
// results are bit-identical to round 1's kernel; the scalar stage and store (still taken for odd
// shapes) ARE round 1's, and tests/test_post_simt.py compares the two paths bit for bit.
#include <algorithm>

#include "common.cuh"

namespace kbmod {

constexpr int PSF_TABLE_FLOATS = 8000;      // 32 000 bytes: the kernel parameter space holds 32 764
struct PsfTable {
    float t[PSF_TABLE_FLOATS];              // images of one launch, P*P floats each
};

constexpr int TILE_W = 64;
constexpr int TILE_H = 32;
constexpr int STRIP = 8;
constexpr int PSI_THREADS = (TILE_W / STRIP) * TILE_H;   // 256

template <int R>
struct PsiPhiGeom {
    static constexpr int P = 2 * R + 1;
    static constexpr int NV4 = (STRIP + 2 * R + 3) / 4;           // float4 loads per window
    static constexpr int PITCH4_RAW = (TILE_W - STRIP) / 4 + NV4;
    static constexpr int PITCH4 = (PITCH4_RAW % 2) ? PITCH4_RAW : PITCH4_RAW + 1;   // odd
    static constexpr int PITCH = 4 * PITCH4;                      // floats
    static constexpr int ROWS = TILE_H + 2 * R;
    static constexpr int COLS = TILE_W + 2 * R;                   // staged columns that matter
    static constexpr int PP4 = (P + 3) / 4 * 4;                   // padded PSF row
    static constexpr size_t SMEM = sizeof(float) * (2 * ROWS * PITCH + 2 * P * PP4);
    static_assert(2 * ROWS * PITCH >= 2 * TILE_W * TILE_H, "the output tile is staged in the s/w planes");
};

// S1 for one pixel: (s, w) = (sci/var, 1/var) on a good pixel, (0, 0) otherwise
__device__ __forceinline__ void weigh(float sc, float va, bool masked, float& s, float& w) {
    // finite(sc) && finite(va) && va > 0
    if (!masked && fabsf(sc) <= 3.402823466e38f && va > 0.0f && va <= 3.402823466e38f) {
        w = __fdiv_rn(1.0f, va);
        s = __fdiv_rn(sc, va);
    } else {
        s = 0.0f; w = 0.0f;
    }
}

template <int R, bool VEC>
__global__ void __launch_bounds__(PSI_THREADS)
psi_phi_kernel(const float* __restrict__ sci_all, const float* __restrict__ var_all,
               const uint8_t* __restrict__ mask_all, int H, int W, int tiles_x, int tiles, int img0,
               float2* __restrict__ out_all, const __grid_constant__ PsfTable psf) {
    using G = PsiPhiGeom<R>;
    constexpr int P = G::P;
    extern __shared__ __align__(16) unsigned char smem_raw[];
    float* s_pl = reinterpret_cast<float*>(smem_raw);
    float* w_pl = s_pl + G::ROWS * G::PITCH;
    float* t_pl = w_pl + G::ROWS * G::PITCH;
    float* t2_pl = t_pl + P * G::PP4;

    const int tid = threadIdx.x;
    const int img_l = blockIdx.x / tiles, tile = blockIdx.x - img_l * tiles;   // image within this launch
    const int x_tile = (tile % tiles_x) * TILE_W;
    const int y_tile = (tile / tiles_x) * TILE_H;
    const size_t img_off = (size_t)(img0 + img_l) * H * W;
    const float* __restrict__ sci = sci_all + img_off;
    const float* __restrict__ var = var_all + img_off;
    const uint8_t* __restrict__ mask = mask_all ? mask_all + img_off : nullptr;
    float2* __restrict__ out = out_all + img_off;
    const float* T = psf.t + img_l * (P * P);

    // PSF and PSF^2 rows, zero padded to a multiple of 4
    for (int k = tid; k < P * G::PP4; k += PSI_THREADS) {
        const int dy = k / G::PP4, dx = k - dy * G::PP4;
        const float t = (dx < P) ? T[dy * P + dx] : 0.0f;
        t_pl[k] = t;
        t2_pl[k] = t * t;
    }
    // S1: weights of tile + halo (zero outside the image, on masked or unusable pixels)
    if constexpr (VEC) {
        // groups of 4 pixels starting at a multiple of 4: with W % 4 == 0 a group is inside the image
        // or outside it as a whole, and its loads are 16-byte (mask: 4-byte) aligned
        const int x_al = (x_tile - R) & ~3, off = (x_tile - R) - x_al;
        const int ngroups = (G::PITCH + off + 3) / 4;
        for (int k = tid; k < G::ROWS * ngroups; k += PSI_THREADS) {
            const int ry = k / ngroups, g = k - ry * ngroups;
            const int gy = y_tile + ry - R, gx = x_al + 4 * g;
            float s[4] = {0.0f, 0.0f, 0.0f, 0.0f}, w[4] = {0.0f, 0.0f, 0.0f, 0.0f};
            if (gy >= 0 && gy < H && gx >= 0 && gx < W) {
                const size_t p = (size_t)gy * W + gx;
                const float4 sc = __ldg(reinterpret_cast<const float4*>(sci + p));
                const float4 va = __ldg(reinterpret_cast<const float4*>(var + p));
                const unsigned m = mask ? __ldg(reinterpret_cast<const unsigned*>(mask + p)) : 0u;
                weigh(sc.x, va.x, (m & 0x000000FFu) != 0, s[0], w[0]);
                weigh(sc.y, va.y, (m & 0x0000FF00u) != 0, s[1], w[1]);
                weigh(sc.z, va.z, (m & 0x00FF0000u) != 0, s[2], w[2]);
                weigh(sc.w, va.w, (m & 0xFF000000u) != 0, s[3], w[3]);
            }
#pragma unroll
            for (int e = 0; e < 4; ++e) {
                const int rx = 4 * g + e - off;
                if (rx >= 0 && rx < G::PITCH) {
                    const bool used = rx < G::COLS;          // the pad columns of the pitch stay zero
                    s_pl[ry * G::PITCH + rx] = used ? s[e] : 0.0f;
                    w_pl[ry * G::PITCH + rx] = used ? w[e] : 0.0f;
                }
            }
        }
    } else {
        for (int k = tid; k < G::ROWS * G::PITCH; k += PSI_THREADS) {
            const int ry = k / G::PITCH, rx = k - ry * G::PITCH;
            const int gy = y_tile + ry - R, gx = x_tile + rx - R;
            float s = 0.0f, w = 0.0f;
            if (rx < G::COLS && gy >= 0 && gy < H && gx >= 0 && gx < W) {
                const size_t g = (size_t)gy * W + gx;
                weigh(__ldg(sci + g), __ldg(var + g), mask ? (__ldg(mask + g) != 0) : false, s, w);
            }
            s_pl[k] = s;
            w_pl[k] = w;
        }
    }
    __syncthreads();

    // lane -> (strip, row): a quarter warp = 4 strips x 2 rows
    const int lane = tid & 31, warp = tid >> 5;
    const int tx = (lane & 3) | (((lane >> 3) & 1) << 2);
    const int ty = warp * 4 + (((lane >> 2) & 1) | (((lane >> 4) & 1) << 1));

    float psi[STRIP], phi[STRIP];
#pragma unroll
    for (int k = 0; k < STRIP; ++k) psi[k] = phi[k] = 0.0f;

#pragma unroll 1
    for (int dy = 0; dy < P; ++dy) {
        const float4* srow = reinterpret_cast<const float4*>(s_pl + (ty + dy) * G::PITCH + tx * STRIP);
        const float4* wrow = reinterpret_cast<const float4*>(w_pl + (ty + dy) * G::PITCH + tx * STRIP);
        const float4* trow = reinterpret_cast<const float4*>(t_pl + dy * G::PP4);
        const float4* t2row = reinterpret_cast<const float4*>(t2_pl + dy * G::PP4);
        float sv[4 * G::NV4], wv[4 * G::NV4];
#pragma unroll
        for (int k = 0; k < G::NV4; ++k) {
            const float4 a = srow[k], b = wrow[k];
            sv[4 * k] = a.x; sv[4 * k + 1] = a.y; sv[4 * k + 2] = a.z; sv[4 * k + 3] = a.w;
            wv[4 * k] = b.x; wv[4 * k + 1] = b.y; wv[4 * k + 2] = b.z; wv[4 * k + 3] = b.w;
        }
#pragma unroll
        for (int q = 0; q < G::PP4 / 4; ++q) {
            const float4 t4 = trow[q], u4 = t2row[q];
            const float tt[4] = {t4.x, t4.y, t4.z, t4.w};
            const float uu[4] = {u4.x, u4.y, u4.z, u4.w};
#pragma unroll
            for (int e = 0; e < 4; ++e) {
                const int dx = 4 * q + e;
                if (dx < P) {
#pragma unroll
                    for (int k = 0; k < STRIP; ++k) {
                        psi[k] = fmaf(sv[k + dx], tt[e], psi[k]);
                        phi[k] = fmaf(wv[k + dx], uu[e], phi[k]);
                    }
                }
            }
        }
    }

    // validity of the centre pixels, then the outputs: straight to global memory (scalar path) or
    // through shared memory so that consecutive lanes store consecutive 16-byte vectors
    const float nan = __int_as_float(0x7fc00000);
    const float* wc = w_pl + (ty + R) * G::PITCH + tx * STRIP + R;
    float2 o[STRIP];
#pragma unroll
    for (int k = 0; k < STRIP; ++k) {
        const bool ok = (wc[k] > 0.0f) && (phi[k] > 0.0f);
        o[k] = ok ? make_float2(psi[k], phi[k]) : make_float2(nan, 0.0f);
    }
    if constexpr (VEC) {
        __syncthreads();                                  // every thread is done with the s / w planes
        float4* tile4 = reinterpret_cast<float4*>(smem_raw);       // [TILE_H][TILE_W / 2] pairs of pixels
#pragma unroll
        for (int k = 0; k < STRIP; k += 2)
            tile4[ty * (TILE_W / 2) + tx * (STRIP / 2) + k / 2] = make_float4(o[k].x, o[k].y, o[k + 1].x, o[k + 1].y);
        __syncthreads();
#pragma unroll
        for (int pass = 0; pass < (TILE_W / 2) * TILE_H / PSI_THREADS; ++pass) {
            const int idx = pass * PSI_THREADS + tid;
            const int row = idx / (TILE_W / 2), c2 = idx - row * (TILE_W / 2);
            const int gy = y_tile + row, gx = x_tile + 2 * c2;
            if (gy < H && gx < W)                          // W is even here: the pair is inside as a whole
                *reinterpret_cast<float4*>(out + (size_t)gy * W + gx) = tile4[idx];
        }
    } else {
        const int gy = y_tile + ty;
        if (gy < H) {
            const int gx0 = x_tile + tx * STRIP;
            float2* orow = out + (size_t)gy * W + gx0;
#pragma unroll
            for (int k = 0; k < STRIP; ++k)
                if (gx0 + k < W) orow[k] = o[k];
        }
    }
}

template <int R>
static int launch_r(const float* sci, const float* var, const uint8_t* mask, const float* psf_host,
                    int N, int H, int W, float2* psiphi, cudaStream_t st) {
    using G = PsiPhiGeom<R>;
    // vector I/O needs whole 4-pixel groups per row and aligned bases (image planes then stay aligned)
    const bool vec = (W % 4 == 0) && !((uintptr_t)sci & 15) && !((uintptr_t)var & 15) && !((uintptr_t)mask & 3) &&
                     !((uintptr_t)psiphi & 15);
    auto kern = vec ? psi_phi_kernel<R, true> : psi_phi_kernel<R, false>;
    if (cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)G::SMEM) != cudaSuccess)
        return KBMOD_ERR_CUDA;
    const int tiles_x = (W + TILE_W - 1) / TILE_W, tiles_y = (H + TILE_H - 1) / TILE_H;
    const long long tiles = (long long)tiles_x * tiles_y;
    constexpr int PER_LAUNCH = PSF_TABLE_FLOATS / (G::P * G::P);
    if (tiles * std::min(N, PER_LAUNCH) > 0x7FFFFFFFLL) return KBMOD_ERR_UNSUPPORTED;
    PsfTable table;
    for (int i0 = 0; i0 < N; i0 += PER_LAUNCH) {
        const int n = std::min(PER_LAUNCH, N - i0);
        for (int k = 0; k < n * G::P * G::P; ++k) table.t[k] = psf_host[(size_t)i0 * G::P * G::P + k];
        for (int k = n * G::P * G::P; k < PSF_TABLE_FLOATS; ++k) table.t[k] = 0.0f;
        KBMOD_LAUNCH(kern, (unsigned)(tiles * n), PSI_THREADS, G::SMEM, st, sci, var, mask, H, W, tiles_x, (int)tiles,
                     i0, psiphi, table);
        note_launch();
    }
    return cudaGetLastError() == cudaSuccess ? KBMOD_OK : KBMOD_ERR_CUDA;
}

int launch_psi_phi(const float* sci, const float* var, const uint8_t* mask, const float* psf_host,
                   int N, int H, int W, int P, float2* psiphi, cudaStream_t st) {
    switch ((P - 1) / 2) {
#define KB_CASE(R) case R: return launch_r<R>(sci, var, mask, psf_host, N, H, W, psiphi, st);
        KB_CASE(0) KB_CASE(1) KB_CASE(2) KB_CASE(3) KB_CASE(4) KB_CASE(5) KB_CASE(6) KB_CASE(7)
        KB_CASE(8) KB_CASE(9) KB_CASE(10) KB_CASE(11) KB_CASE(12) KB_CASE(13) KB_CASE(14) KB_CASE(15)
#undef KB_CASE
    }
    return KBMOD_ERR_UNSUPPORTED;
}

}  // namespace kbmod
