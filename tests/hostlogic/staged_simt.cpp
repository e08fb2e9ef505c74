// tests/hostlogic/staged_simt.cpp -- TEST INFRASTRUCTURE.  Compiles csrc/search_staged.cu with g++
// against the SIMT emulator of tests/hostlogic/simt/ and exposes launch_search_staged (host plan,
// tensor maps, encode kernel, the persistent producer/consumer kernel) as a C function over HOST
// memory, so that tests/test_staged_simt.py can compare the kernel's device-side logic with the
// oracle without a GPU.  Built by the test with
//   g++ -O1 -std=c++17 -ffp-contract=off -shared -fPIC -Itests/hostlogic/simt -Iinclude
//       -Ipaper_1901_02492_b200/csrc -DKBMOD_SIMT_EMUL='"simt_ptx.h"' tests/hostlogic/staged_simt.cpp
#include <cuda.h>
#include <cuda_runtime.h>
#include <devmem.h>

namespace kbmod {
alignas(1024) unsigned char smem_raw[simt::SMEM_MAX + 64];
}  // namespace kbmod

#include "search_staged.cu"

namespace kbmod {
void note_launch(int) {}
}  // namespace kbmod

extern "C" {

// stats[0..5] = shared-memory faults, TMA loads, TMA alignment faults, kernel launches, status word, plan entries
// Result planes hold the band [y_begin, y_end) only.  geom = kbmod_search_options.staged_geom.
int simt_search_staged(const float* psiphi, const double* times, int N, int H, int W, const float* vel_grid, int V,
                       int K, int min_obs, int y_begin, int y_end, int32_t* vel_idx, int32_t* n_obs, float* psi,
                       float* phi, float* nu, float* alpha, int geom, int order, unsigned seed, int sms, int tma_delay,
                       long long* stats) {
    using namespace kbmod;
    simt::cfg().order = order;
    simt::cfg().seed = seed;
    simt::cfg().sms = sms;
    simt::cfg().tma_delay = tma_delay;
    simt::State& s = simt::S();
    s.smem = smem_raw;
    s.smem_faults = s.tma_loads = s.tma_faults = s.launches = 0;
    DtTable dt;
    for (int i = 0; i < KBMOD_MAX_IMAGES; ++i) dt.dt[i] = 0.0f;
    for (int i = 0; i < N; ++i) dt.dt[i] = (float)(times[i] - times[0]);
    // every buffer the kernels see is its own heap block of exactly the size the product gives them
    // (devmem.h): inputs copied in, result planes copied back
    const size_t npix = (size_t)N * H * W, nres = (size_t)(y_end - y_begin) * W * K;
    simt::DevBuf d_pp(psiphi, npix * 8), d_vel(vel_grid, (size_t)V * 8);
    simt::DevBuf d_plan(staged_plan_bytes(N, V)), d_enc(staged_enc_bytes(N, H, W)), d_status(sizeof(int));
    simt::DevBuf d_vi(nres * 4), d_no(nres * 4), d_psi(nres * 4), d_phi(nres * 4), d_nu(nres * 4), d_al(nres * 4);
    kbmod_result out{d_vi.as<int32_t>(), d_no.as<int32_t>(), d_psi.as<float>(), d_phi.as<float>(),
                     d_nu.as<float>(), d_al.as<float>()};
    const int rc = launch_search_staged(d_pp.as<const float2>(), dt, N, H, W, vel_grid, V, K, min_obs, y_begin, y_end,
                                        out, d_plan.p, d_vel.as<const float2>(), d_enc.as<float2>(),
                                        d_status.as<int>(), geom, nullptr);
    d_vi.copy_to(vel_idx); d_no.copy_to(n_obs); d_psi.copy_to(psi); d_phi.copy_to(phi); d_nu.copy_to(nu);
    d_al.copy_to(alpha);
    const int status = *d_status.as<int>();
    stats[0] = s.smem_faults; stats[1] = s.tma_loads; stats[2] = s.tma_faults; stats[3] = s.launches;
    stats[4] = status; stats[5] = 0;
    return rc;
}

}  // extern "C"
