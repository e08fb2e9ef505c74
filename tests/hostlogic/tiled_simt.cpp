// tests/hostlogic/tiled_simt.cpp -- TEST INFRASTRUCTURE.  Compiles csrc/search_tiled.cu with g++
// against the SIMT emulator of tests/hostlogic/simt/ and exposes launch_search_tiled (host plan,
// encode kernel, search_tiled_kernel or search_tiledq_kernel) as a C function over HOST memory
// (tests/test_tiled_simt.py).  search_tiled_kernel is validated on B200 hardware, so its run under
// emulation also checks the emulator; search_tiledq_kernel's logic is checked here first.  Built with
//   g++ -O1 -std=c++17 -ffp-contract=off -shared -fPIC -Itests/hostlogic/simt -Iinclude
//       -Ipaper_1901_02492_b200/csrc -DKBMOD_SIMT_EMUL=1 tests/hostlogic/tiled_simt.cpp
#include <cuda.h>
#include <cuda_runtime.h>
#include <devmem.h>

namespace kbmod {
alignas(1024) unsigned char smem_raw[simt::SMEM_MAX + 64];
}  // namespace kbmod

#include "search_tiled.cu"

namespace kbmod {
void note_launch(int) {}
}  // namespace kbmod

extern "C" {

// stats[0..4] = shared-memory faults (none possible here: plain pointers), 0, 0, kernel launches, 0
// Result planes hold the band [y_begin, y_end) only.  group_w = kbmod_search_options.tile_group_w.
int simt_search_tiled(const float* psiphi, const double* times, int N, int H, int W, const float* vel_grid, int V,
                      int K, int min_obs, int y_begin, int y_end, int32_t* vel_idx, int32_t* n_obs, float* psi,
                      float* phi, float* nu, float* alpha, int queued, int group_w, int order, unsigned seed,
                      long long* stats) {
    using namespace kbmod;
    simt::cfg().order = order;
    simt::cfg().seed = seed;
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
    simt::DevBuf d_plan(tiled_plan_bytes(N, V, K)), d_enc((size_t)N * H * enc_pitch(W) * 8);
    simt::DevBuf d_vi(nres * 4), d_no(nres * 4), d_psi(nres * 4), d_phi(nres * 4), d_nu(nres * 4), d_al(nres * 4);
    kbmod_result out{d_vi.as<int32_t>(), d_no.as<int32_t>(), d_psi.as<float>(), d_phi.as<float>(),
                     d_nu.as<float>(), d_al.as<float>()};
    const int rc = launch_search_tiled(d_pp.as<const float2>(), dt, N, H, W, vel_grid, V, K, min_obs, y_begin, y_end,
                                       out, d_plan.p, d_vel.as<const float2>(), d_enc.as<float2>(), queued != 0,
                                       group_w, nullptr);
    d_vi.copy_to(vel_idx); d_no.copy_to(n_obs); d_psi.copy_to(psi); d_phi.copy_to(phi); d_nu.copy_to(nu);
    d_al.copy_to(alpha);
    stats[0] = s.smem_faults; stats[1] = 0; stats[2] = 0; stats[3] = s.launches; stats[4] = 0;
    return rc;
}

// Threshold mode on the queued kernel (kbmod_search_threshold with kernel 4).  Returns the count.
long long simt_search_tiled_threshold(const float* psiphi, const double* times, int N, int H, int W,
                                      const float* vel_grid, int V, int min_obs, float nu_min, int y_begin, int y_end,
                                      long long capacity, int32_t* x, int32_t* y, int32_t* vel_idx, int32_t* n_obs,
                                      float* psi, float* phi, float* nu, float* alpha, int order, unsigned seed) {
    using namespace kbmod;
    simt::cfg().order = order;
    simt::cfg().seed = seed;
    simt::State& s = simt::S();
    s.smem = smem_raw;
    s.smem_faults = s.launches = 0;
    DtTable dt;
    for (int i = 0; i < KBMOD_MAX_IMAGES; ++i) dt.dt[i] = 0.0f;
    for (int i = 0; i < N; ++i) dt.dt[i] = (float)(times[i] - times[0]);
    const size_t npix = (size_t)N * H * W, nc = (size_t)capacity * 4;
    simt::DevBuf d_pp(psiphi, npix * 8), d_vel(vel_grid, (size_t)V * 8), d_count(8);
    simt::DevBuf d_plan(tiled_plan_bytes(N, V, 8)), d_enc((size_t)N * H * enc_pitch(W) * 8);
    simt::DevBuf d_x(nc), d_y(nc), d_vi(nc), d_no(nc), d_psi(nc), d_phi(nc), d_nu(nc), d_al(nc);
    *d_count.as<unsigned long long>() = 0;
    kbmod_candidates out{d_x.as<int32_t>(), d_y.as<int32_t>(), d_vi.as<int32_t>(), d_no.as<int32_t>(), d_psi.as<float>(),
                         d_phi.as<float>(), d_nu.as<float>(), d_al.as<float>()};
    TiledPlan plan;
    if (int rc = tiled_plan_build(dt, N, H, W, vel_grid, V, 8, true, plan)) return rc;
    const int rc = tiled_launch_threshold(plan, d_pp.as<const float2>(), dt, N, H, W, min_obs, nu_min, y_begin, y_end, out,
                                          (unsigned long long)capacity, d_count.as<unsigned long long>(), d_plan.p,
                                          d_vel.as<const float2>(), d_enc.as<float2>(), 0, nullptr);
    if (rc) return rc;
    d_x.copy_to(x); d_y.copy_to(y); d_vi.copy_to(vel_idx); d_no.copy_to(n_obs); d_psi.copy_to(psi); d_phi.copy_to(phi);
    d_nu.copy_to(nu); d_al.copy_to(alpha);
    return (long long)*d_count.as<unsigned long long>();
}

// launch_search_tiled's own size limits (int16 shift encoding, int32 element offsets): the launch
// must refuse, before touching any buffer, a stack whose (N+1)*H*W element offsets do not fit int32
int simt_tiled_limits(int N, int H, int W, int V, int K) {
    using namespace kbmod;
    DtTable dt;
    for (int i = 0; i < KBMOD_MAX_IMAGES; ++i) dt.dt[i] = (float)i;
    std::vector<float> vel((size_t)2 * V, 1.0f);
    kbmod_result out{nullptr, nullptr, nullptr, nullptr, nullptr, nullptr};
    return launch_search_tiled(nullptr, dt, N, H, W, vel.data(), V, K, 1, 0, H, out, nullptr, nullptr, nullptr, true, 0,
                               nullptr);
}

// Detector self-test: reads the element `past` elements beyond a 64-byte emulated device buffer
// through __ldg.  past = 0 is legal; past = 1 must abort under AddressSanitizer.
unsigned long long simt_selftest_ldg_past_end(int past) {
    simt::DevBuf b(64);
    return __ldg(b.as<const unsigned long long>() + 7 + past);
}

// Detector self-test: a float4 load `misalign` bytes off a 16-byte boundary, inside the buffer.
// misalign = 0 is legal; 4 or 8 is a misaligned-address fault on the GPU and must abort under UBSan.
float simt_selftest_ldg128_misaligned(int misalign) {
    simt::DevBuf b(64, 256, 0);
    const float4 v = __ldg(reinterpret_cast<const float4*>(b.as<char>() + 16 + misalign));
    return v.x + v.w;
}

}  // extern "C"
