// common.cuh -- shared declarations of the CUDA path (internal; not part of the C ABI).
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>
#include <stddef.h>
#include "kbmod_b200.h"

// Kernel launch.  The SIMT-emulation test build (tests/hostlogic/simt/, g++, no GPU) runs the
// kernel's CTAs on the CPU instead; the product build is the plain triple-chevron launch.
#if defined(KBMOD_SIMT_EMUL)
#define KBMOD_LAUNCH(kern, grid, block, smem, stream, ...) ::simt::launch(kern, ::simt::as_dim3(grid), ::simt::as_dim3(block), (size_t)(smem), __VA_ARGS__)
#else
#define KBMOD_LAUNCH(kern, grid, block, smem, stream, ...) kern<<<(grid), (block), (smem), (stream)>>>(__VA_ARGS__)
#endif

namespace kbmod {

// every kernel launch of the library goes through this counter (kbmod_launch_count()).
void note_launch(int n = 1);

struct DtTable {                 // dt_i = (float)(times[i] - times[0]); passed by value
    float dt[KBMOD_MAX_IMAGES];
};

// ---- psi/phi builder (psi_phi.cu)
int launch_psi_phi(const float* sci, const float* var, const uint8_t* mask, const float* psf_host,
                   int N, int H, int W, int P, float2* psiphi, cudaStream_t st);

// ---- direct-gather search (search_direct.cu): any shape, global loads through L1/L2
int launch_search_direct(const float2* psiphi, const DtTable& dt, int N, int H, int W,
                         const float2* vel_dev, int V, int K, int min_obs, int y_begin, int y_end,
                         const kbmod_result& out, cudaStream_t st);
int launch_search_direct_threshold(const float2* psiphi, const DtTable& dt, int N, int H, int W,
                                   const float2* vel_dev, int V, int min_obs, float nu_min, int y_begin, int y_end,
                                   const kbmod_candidates& out, unsigned long long capacity,
                                   unsigned long long* count, cudaStream_t st);
int launch_eval_trajectories(const float2* psiphi, const DtTable& dt, int N, int H, int W,
                             const int32_t* x0y0, const float2* vxvy, int M, float* Psi,
                             float* Phi, int32_t* n_obs, int32_t* ixiy, cudaStream_t st);
int launch_interleave(const float* psi, const float* phi, size_t n, float2* out, cudaStream_t st);

// ---- rows around the search (postproc.cu): N1 light-curve filter, N2 stamps + moments, N3 mask builder
int launch_filter_candidates(const float2* psiphi, const DtTable& dt, int N, int H, int W, const int32_t* x0y0,
                             const float2* vxvy, int M, float sigma_reject, float q, float* psi, float* phi,
                             int32_t* n_obs, float* nu, float* alpha, unsigned long long* keep, float2* kalman,
                             cudaStream_t st);
int launch_coadd_stamps(const float* sci, const uint8_t* mask, const DtTable& dt, int N, int H, int W,
                        const int32_t* x0y0, const float2* vxvy, const unsigned long long* keep, int M, int R,
                        float* stamps, float* moments, cudaStream_t st);
int launch_build_mask(const float* sci, const float* var, const uint8_t* mask_in, int N, int H, int W,
                      float sigma_thr, int grow, int min_images, float bright_counts, uint8_t* mask_out,
                      cudaStream_t st);

size_t cluster_workspace_bytes(int M);
int launch_cluster_candidates(const int32_t* x0y0, const float2* vxvy, const float* nu, int M, float eps_xy,
                              float eps_v, int min_samples, int32_t* label, uint8_t* rep, void* workspace,
                              cudaStream_t st);

// ---- S3: the trajectory pixel, exactly as include/kbmod_b200.h states it
__device__ __forceinline__ bool traj_pixel(int p0, float v, float dt, int n, int& ip) {
    const float f = __fadd_rn(__int2float_rn(p0), __fmul_rn(v, dt));
    const float g = floorf(__fadd_rn(f, 0.5f));
    if (!(g >= 0.0f && g < (float)n)) return false;
    ip = (int)g;
    return true;
}

// ---- S5
__device__ __forceinline__ float score_nu(float Psi, float Phi) {
    return __fdiv_rn(Psi, __fsqrt_rn(Phi));
}
__device__ __forceinline__ float score_alpha(float Psi, float Phi) { return __fdiv_rn(Psi, Phi); }

}  // namespace kbmod
