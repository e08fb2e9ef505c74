// search_direct.cu -- S3..S6 with direct global gathers (any shape).  The general path and the
// baseline the shared-memory staged kernel (search_staged.cu) is measured against.
//
// One thread = one start pixel; a warp = 32 x-adjacent start pixels, so for a given (velocity,
// image) the warp reads 32 contiguous float2 samples ("horizontally adjacent
// trajectories access them contiguously").  Velocities are visited in index order, images in
// order 0..N-1 with __fadd_rn, so Psi/Phi equal an in-order fp32 sum bit for bit.  The per-pixel
// top-K is a sorted register list; (nu, vel_idx) of the K best are kept and their Psi/Phi/n_obs
// are re-evaluated once at the end.
#include "common.cuh"
#include "topk_list.h"

namespace kbmod {

struct Coadd {
    float Psi, Phi;
    int n;
};

// S3 + S4 for one trajectory (Eq.24-25; validity P:171)
__device__ __forceinline__ Coadd coadd_direct(const float2* __restrict__ psiphi, const DtTable& dt,
                                              int N, int H, int W, int x0, int y0, float vx,
                                              float vy, int32_t* ixiy) {
    Coadd c{0.0f, 0.0f, 0};
    for (int i = 0; i < N; ++i) {
        int ix = -1, iy = -1;
        const bool inx = traj_pixel(x0, vx, dt.dt[i], W, ix);
        const bool iny = traj_pixel(y0, vy, dt.dt[i], H, iy);
        const bool inb = inx && iny;
        if (ixiy) {
            ixiy[2 * i] = inb ? ix : -1;
            ixiy[2 * i + 1] = inb ? iy : -1;
        }
        if (inb) {
            const float2 s = __ldg(psiphi + ((size_t)i * H + iy) * W + ix);
            if (s.x == s.x) {
                c.Psi = __fadd_rn(c.Psi, s.x);
                c.Phi = __fadd_rn(c.Phi, s.y);
                ++c.n;
            }
        }
    }
    return c;
}

template <int KMAX>
__global__ void __launch_bounds__(256)
search_direct_kernel(const float2* __restrict__ psiphi, const __grid_constant__ DtTable dt, int N,
                     int H, int W, const float2* __restrict__ vel, int V, int K, int min_obs,
                     int y_begin, int y_end, kbmod_result out) {
    const int x0 = blockIdx.x * 32 + threadIdx.x;
    const int y0 = y_begin + blockIdx.y * 8 + threadIdx.y;
    if (x0 >= W || y0 >= y_end) return;

    float best_nu[KMAX];
    int best_j[KMAX];
#pragma unroll
    for (int k = 0; k < KMAX; ++k) {
        best_nu[k] = (k < K) ? -INFINITY : INFINITY;        // slots beyond K are never displaced
        best_j[k] = (k < K) ? LIST_EMPTY_IDX : -1;
    }

    for (int j = 0; j < V; ++j) {
        const float2 v = __ldg(vel + j);
        const Coadd c = coadd_direct(psiphi, dt, N, H, W, x0, y0, v.x, v.y, nullptr);
        if (c.n >= min_obs && c.Phi > 0.0f) {
            float nu = score_nu(c.Psi, c.Phi);
            {
                // sorted insert by the rule of topk_list.h (larger nu first, ties: smaller index; an
                // empty slot ranks last, so a candidate with nu = -inf still enters an empty slot)
                int jj = j;
                bool shifting = false;          // after the insert the tail shifts down as is
#pragma unroll
                for (int k = 0; k < KMAX; ++k) {
                    if (shifting || better(nu, jj, best_nu[k], best_j[k])) {
                        shifting = true;
                        const float tn = best_nu[k];
                        const int tj = best_j[k];
                        best_nu[k] = nu;
                        best_j[k] = jj;
                        nu = tn;
                        jj = tj;
                    }
                }
            }
        }
    }

    const size_t base = ((size_t)(y0 - y_begin) * W + x0) * K;
#pragma unroll
    for (int k = 0; k < KMAX; ++k) {
        if (k < K) {
            const int j = best_j[k];
            if (j != LIST_EMPTY_IDX) {
                const float2 v = __ldg(vel + j);
                const Coadd c = coadd_direct(psiphi, dt, N, H, W, x0, y0, v.x, v.y, nullptr);
                out.vel_idx[base + k] = j;
                out.n_obs[base + k] = c.n;
                out.psi[base + k] = c.Psi;
                out.phi[base + k] = c.Phi;
                out.nu[base + k] = score_nu(c.Psi, c.Phi);
                out.alpha[base + k] = score_alpha(c.Psi, c.Phi);
            } else {
                out.vel_idx[base + k] = -1;
                out.n_obs[base + k] = 0;
                out.psi[base + k] = 0.0f;
                out.phi[base + k] = 0.0f;
                out.nu[base + k] = -INFINITY;
                out.alpha[base + k] = 0.0f;
            }
        }
    }
}

int launch_search_direct(const float2* psiphi, const DtTable& dt, int N, int H, int W,
                         const float2* vel_dev, int V, int K, int min_obs, int y_begin, int y_end,
                         const kbmod_result& out, cudaStream_t st) {
    if (y_end <= y_begin) return KBMOD_OK;
    const dim3 block(32, 8);
    const dim3 grid((W + 31) / 32, (y_end - y_begin + 7) / 8);
    if (grid.y > 65535u) return KBMOD_ERR_UNSUPPORTED;
    if (K <= 4)
        KBMOD_LAUNCH(search_direct_kernel<4>, grid, block, 0, st, psiphi, dt, N, H, W, vel_dev, V, K, min_obs, y_begin, y_end, out);
    else if (K <= 8)
        KBMOD_LAUNCH(search_direct_kernel<8>, grid, block, 0, st, psiphi, dt, N, H, W, vel_dev, V, K, min_obs, y_begin, y_end, out);
    else if (K <= 16)
        KBMOD_LAUNCH(search_direct_kernel<16>, grid, block, 0, st, psiphi, dt, N, H, W, vel_dev, V, K, min_obs, y_begin, y_end, out);
    else
        KBMOD_LAUNCH(search_direct_kernel<32>, grid, block, 0, st, psiphi, dt, N, H, W, vel_dev, V, K, min_obs, y_begin, y_end, out);
    note_launch();
    return cudaGetLastError() == cudaSuccess ? KBMOD_OK : KBMOD_ERR_CUDA;
}

// N4: the paper's own retention rule ("examine those that are above a desired detection
// threshold"): every eligible trajectory with nu >= nu_min is appended to a compacted list.
// Same S3/S4/S5 as above; the list order is unspecified (one atomic counter), its content is not.
__global__ void __launch_bounds__(256)
search_direct_threshold_kernel(const float2* __restrict__ psiphi, const __grid_constant__ DtTable dt, int N,
                               int H, int W, const float2* __restrict__ vel, int V, int min_obs, float nu_min,
                               int y_begin, int y_end, kbmod_candidates out, unsigned long long capacity,
                               unsigned long long* count) {
    const int x0 = blockIdx.x * 32 + (threadIdx.x & 31);
    const int y0 = y_begin + blockIdx.y * 8 + (threadIdx.x >> 5);
    if (x0 >= W || y0 >= y_end) return;
    for (int j = 0; j < V; ++j) {
        const float2 v = __ldg(vel + j);
        const Coadd c = coadd_direct(psiphi, dt, N, H, W, x0, y0, v.x, v.y, nullptr);
        if (c.n >= min_obs && c.Phi > 0.0f) {
            const float nu = score_nu(c.Psi, c.Phi);
            if (nu >= nu_min) {
                const unsigned long long slot = atomicAdd(count, 1ull);
                if (slot < capacity) {
                    out.x[slot] = x0; out.y[slot] = y0; out.vel_idx[slot] = j; out.n_obs[slot] = c.n;
                    out.psi[slot] = c.Psi; out.phi[slot] = c.Phi; out.nu[slot] = nu;
                    out.alpha[slot] = score_alpha(c.Psi, c.Phi);
                }
            }
        }
    }
}

int launch_search_direct_threshold(const float2* psiphi, const DtTable& dt, int N, int H, int W,
                                   const float2* vel_dev, int V, int min_obs, float nu_min, int y_begin, int y_end,
                                   const kbmod_candidates& out, unsigned long long capacity,
                                   unsigned long long* count, cudaStream_t st) {
    if (y_end <= y_begin) return KBMOD_OK;
    const dim3 grid((W + 31) / 32, (y_end - y_begin + 7) / 8);
    if (grid.y > 65535u) return KBMOD_ERR_UNSUPPORTED;
    KBMOD_LAUNCH(search_direct_threshold_kernel, grid, 256, 0, st, psiphi, dt, N, H, W, vel_dev, V, min_obs, nu_min,
                 y_begin, y_end, out, capacity, count);
    note_launch();
    return cudaGetLastError() == cudaSuccess ? KBMOD_OK : KBMOD_ERR_CUDA;
}

__global__ void eval_trajectories_kernel(const float2* __restrict__ psiphi,
                                         const __grid_constant__ DtTable dt, int N, int H, int W,
                                         const int32_t* __restrict__ x0y0,
                                         const float2* __restrict__ vxvy, int M, float* Psi,
                                         float* Phi, int32_t* n_obs, int32_t* ixiy) {
    const int m = blockIdx.x * blockDim.x + threadIdx.x;
    if (m >= M) return;
    const float2 v = vxvy[m];
    const Coadd c = coadd_direct(psiphi, dt, N, H, W, x0y0[2 * m], x0y0[2 * m + 1], v.x, v.y,
                                 ixiy ? ixiy + (size_t)m * N * 2 : nullptr);
    Psi[m] = c.Psi;
    Phi[m] = c.Phi;
    n_obs[m] = c.n;
}

int launch_eval_trajectories(const float2* psiphi, const DtTable& dt, int N, int H, int W,
                             const int32_t* x0y0, const float2* vxvy, int M, float* Psi,
                             float* Phi, int32_t* n_obs, int32_t* ixiy, cudaStream_t st) {
    if (M == 0) return KBMOD_OK;
    KBMOD_LAUNCH(eval_trajectories_kernel, (M + 127) / 128, 128, 0, st, psiphi, dt, N, H, W, x0y0, vxvy, M, Psi, Phi,
                 n_obs, ixiy);
    note_launch();
    return cudaGetLastError() == cudaSuccess ? KBMOD_OK : KBMOD_ERR_CUDA;
}

__global__ void interleave_kernel(const float* __restrict__ psi, const float* __restrict__ phi,
                                  size_t n, float2* __restrict__ out) {
    for (size_t k = (size_t)blockIdx.x * blockDim.x + threadIdx.x; k < n;
         k += (size_t)gridDim.x * blockDim.x)
        out[k] = make_float2(psi[k], phi[k]);
}

int launch_interleave(const float* psi, const float* phi, size_t n, float2* out, cudaStream_t st) {
    KBMOD_LAUNCH(interleave_kernel, 148 * 8, 256, 0, st, psi, phi, n, out);
    note_launch();
    return cudaGetLastError() == cudaSuccess ? KBMOD_OK : KBMOD_ERR_CUDA;
}

}  // namespace kbmod
