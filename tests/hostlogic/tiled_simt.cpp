// tests/hostlogic/tiled_simt.cpp -- TEST INFRASTRUCTURE.  Compiles csrc/search_tiled.cu with g++
// against the SIMT emulator of tests/hostlogic/simt/ and exposes launch_search_tiled (host plan,
// encode kernel, search_tiled_kernel or search_tiledq_kernel) as a C function over HOST memory
// (tests/test_tiled_simt.py).  search_tiled_kernel is validated on B200 hardware, so its run under
// emulation also checks the emulator; search_tiledq_kernel's logic is checked here first.  Built with
//   g++ -O1 -std=c++17 -ffp-contract=off -shared -fPIC -Itests/hostlogic/simt -Iinclude
//       -Ipaper_1901_02492_b200/csrc -DKBMOD_SIMT_EMUL=1 tests/hostlogic/tiled_simt.cpp
#include <cuda.h>
#include <cuda_runtime.h>

namespace kbmod {
alignas(1024) unsigned char smem_raw[simt::SMEM_MAX + 64];
}  // namespace kbmod

#include "search_tiled.cu"

namespace kbmod {
void note_launch(int) {}
}  // namespace kbmod

extern "C" {

// stats[0..4] = shared-memory faults (none possible here: plain pointers), 0, 0, kernel launches, 0
int simt_search_tiled(const float* psiphi, const double* times, int N, int H, int W, const float* vel_grid, int V,
                      int K, int min_obs, int32_t* vel_idx, int32_t* n_obs, float* psi, float* phi, float* nu,
                      float* alpha, int queued, int order, unsigned seed, long long* stats) {
    using namespace kbmod;
    simt::cfg().order = order;
    simt::cfg().seed = seed;
    simt::State& s = simt::S();
    s.smem = smem_raw;
    s.smem_faults = s.tma_loads = s.tma_faults = s.launches = 0;
    DtTable dt;
    for (int i = 0; i < KBMOD_MAX_IMAGES; ++i) dt.dt[i] = 0.0f;
    for (int i = 0; i < N; ++i) dt.dt[i] = (float)(times[i] - times[0]);
    kbmod_result out{vel_idx, n_obs, psi, phi, nu, alpha};
    std::vector<unsigned char> plan(tiled_plan_bytes(N, V, K) + 256), enc((size_t)N * H * W * 8 + 512);
    unsigned char* encp = enc.data() + ((256 - ((uintptr_t)enc.data() & 255)) & 255);
    const int rc = launch_search_tiled(reinterpret_cast<const float2*>(psiphi), dt, N, H, W, vel_grid, V, K, min_obs,
                                       out, plan.data(), reinterpret_cast<const float2*>(vel_grid),
                                       reinterpret_cast<float2*>(encp), queued != 0, nullptr);
    stats[0] = s.smem_faults; stats[1] = 0; stats[2] = 0; stats[3] = s.launches; stats[4] = 0;
    return rc;
}

}  // extern "C"
