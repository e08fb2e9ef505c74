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
#include "common.cuh"

namespace kbmod {

struct PsfParam {
    float t[KBMOD_MAX_PSF * KBMOD_MAX_PSF];
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
};

template <int R>
__global__ void __launch_bounds__(PSI_THREADS)
psi_phi_kernel(const float* __restrict__ sci, const float* __restrict__ var,
               const uint8_t* __restrict__ mask, int H, int W, float2* __restrict__ out,
               const __grid_constant__ PsfParam psf) {
    using G = PsiPhiGeom<R>;
    constexpr int P = G::P;
    extern __shared__ __align__(16) float smem[];
    float* s_pl = smem;
    float* w_pl = s_pl + G::ROWS * G::PITCH;
    float* t_pl = w_pl + G::ROWS * G::PITCH;
    float* t2_pl = t_pl + P * G::PP4;

    const int tid = threadIdx.x;
    const int x_tile = blockIdx.x * TILE_W;
    const int y_tile = blockIdx.y * TILE_H;

    // PSF and PSF^2 rows, zero padded to a multiple of 4
    for (int k = tid; k < P * G::PP4; k += PSI_THREADS) {
        const int dy = k / G::PP4, dx = k - dy * G::PP4;
        const float t = (dx < P) ? psf.t[dy * P + dx] : 0.0f;
        t_pl[k] = t;
        t2_pl[k] = t * t;
    }
    // S1: weights of tile + halo (zero outside the image, on masked or unusable pixels)
    for (int k = tid; k < G::ROWS * G::PITCH; k += PSI_THREADS) {
        const int ry = k / G::PITCH, rx = k - ry * G::PITCH;
        const int gy = y_tile + ry - R, gx = x_tile + rx - R;
        float s = 0.0f, w = 0.0f;
        if (rx < G::COLS && gy >= 0 && gy < H && gx >= 0 && gx < W) {
            const size_t g = (size_t)gy * W + gx;
            const float sc = __ldg(sci + g), va = __ldg(var + g);
            const bool m = mask ? (__ldg(mask + g) != 0) : false;
            // finite(sc) && finite(va) && va > 0
            if (!m && fabsf(sc) <= 3.402823466e38f && va > 0.0f && va <= 3.402823466e38f) {
                w = __fdiv_rn(1.0f, va);
                s = __fdiv_rn(sc, va);
            }
        }
        s_pl[k] = s;
        w_pl[k] = w;
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

    const int gy = y_tile + ty;
    if (gy < H) {
        const float* wc = w_pl + (ty + R) * G::PITCH + tx * STRIP + R;
        const int gx0 = x_tile + tx * STRIP;
        float2* orow = out + (size_t)gy * W + gx0;
#pragma unroll
        for (int k = 0; k < STRIP; ++k) {
            if (gx0 + k < W) {
                const bool ok = (wc[k] > 0.0f) && (phi[k] > 0.0f);
                orow[k] = ok ? make_float2(psi[k], phi[k]) : make_float2(__int_as_float(0x7fc00000), 0.0f);
            }
        }
    }
}

template <int R>
static int launch_r(const float* sci, const float* var, const uint8_t* mask, const float* psf_host,
                    int N, int H, int W, float2* psiphi, cudaStream_t st) {
    using G = PsiPhiGeom<R>;
    auto kern = psi_phi_kernel<R>;
    if (cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)G::SMEM) != cudaSuccess)
        return KBMOD_ERR_CUDA;
    const dim3 grid((W + TILE_W - 1) / TILE_W, (H + TILE_H - 1) / TILE_H);
    PsfParam p;
    for (int i = 0; i < N; ++i) {
        for (int k = 0; k < KBMOD_MAX_PSF * KBMOD_MAX_PSF; ++k) p.t[k] = 0.0f;
        for (int k = 0; k < G::P * G::P; ++k) p.t[k] = psf_host[(size_t)i * G::P * G::P + k];
        const size_t off = (size_t)i * H * W;
        kern<<<grid, PSI_THREADS, G::SMEM, st>>>(sci + off, var + off, mask ? mask + off : nullptr,
                                                H, W, psiphi + off, p);
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
