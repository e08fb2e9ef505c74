// tests/hostlogic/post_simt.cpp -- TEST INFRASTRUCTURE.  Compiles csrc/search_direct.cu (the
// direct-gather search in its top-K and threshold forms, the trajectory test hook) and
// csrc/postproc.cu (N1 light-curve filter, N2 stamps and moments, N3 mask builder) with g++ against
// the SIMT emulator of tests/hostlogic/simt/ and exposes their launchers as C functions over HOST
// memory, every buffer an exact-size heap block (devmem.h), so that tests/test_post_simt.py can
// compare the kernels' device-side logic with the oracle bit for bit without a GPU -- also under
// AddressSanitizer (tests/test_simt_sanitized.py).
#include <cuda.h>
#include <cuda_runtime.h>
#include <devmem.h>

namespace kbmod {
alignas(1024) unsigned char smem_raw[simt::SMEM_MAX + 64];
}  // namespace kbmod

#include "search_direct.cu"
#include "postproc.cu"
#include "psi_phi.cu"

namespace kbmod {
void note_launch(int) {}
static DtTable dt_of(const double* times, int N) {
    DtTable dt;
    for (int i = 0; i < KBMOD_MAX_IMAGES; ++i) dt.dt[i] = 0.0f;
    for (int i = 0; i < N; ++i) dt.dt[i] = (float)(times[i] - times[0]);
    return dt;
}
static void prep(int order, unsigned seed) {
    simt::cfg().order = order;
    simt::cfg().seed = seed;
    simt::State& s = simt::S();
    s.smem = smem_raw;
    s.smem_faults = s.tma_loads = s.tma_faults = s.launches = 0;
}
}  // namespace kbmod

extern "C" {
using namespace kbmod;

// S1 + S2.  misalign != 0 hands the kernel a sci plane that is only 4-byte aligned, which selects the
// scalar stage and store (round 1's path) for the same data.  launches = kernel launches issued.
int simt_make_psi_phi(const float* sci, const float* var, const uint8_t* mask, const float* psf, int N, int H, int W,
                      int P, float* psiphi, int misalign, int* launches, int order, unsigned seed) {
    prep(order, seed);
    const size_t npix = (size_t)N * H * W;
    simt::DevBuf d_sci(npix * 4 + (misalign ? 4 : 0)), d_var(var, npix * 4), d_pp(npix * 8);
    float* sci_dev = reinterpret_cast<float*>(d_sci.as<char>() + (misalign ? 4 : 0));
    memcpy(sci_dev, sci, npix * 4);
    simt::DevBuf d_mask(mask ? (const void*)mask : (const void*)sci, mask ? npix : 0);
    const int rc = launch_psi_phi(sci_dev, d_var.as<const float>(), mask ? d_mask.as<const uint8_t>() : nullptr, psf, N, H,
                                  W, P, d_pp.as<float2>(), nullptr);
    d_pp.copy_to(psiphi);
    *launches = (int)simt::S().launches;
    return rc;
}

int simt_search_direct(const float* psiphi, const double* times, int N, int H, int W, const float* vel, int V, int K,
                       int min_obs, int y_begin, int y_end, int32_t* vel_idx, int32_t* n_obs, float* psi, float* phi,
                       float* nu, float* alpha, int order, unsigned seed) {
    prep(order, seed);
    const size_t npix = (size_t)N * H * W, nres = (size_t)(y_end - y_begin) * W * K;
    simt::DevBuf d_pp(psiphi, npix * 8), d_vel(vel, (size_t)V * 8);
    simt::DevBuf d_vi(nres * 4), d_no(nres * 4), d_psi(nres * 4), d_phi(nres * 4), d_nu(nres * 4), d_al(nres * 4);
    kbmod_result out{d_vi.as<int32_t>(), d_no.as<int32_t>(), d_psi.as<float>(), d_phi.as<float>(), d_nu.as<float>(),
                     d_al.as<float>()};
    const int rc = launch_search_direct(d_pp.as<const float2>(), dt_of(times, N), N, H, W, d_vel.as<const float2>(), V, K,
                                        min_obs, y_begin, y_end, out, nullptr);
    d_vi.copy_to(vel_idx); d_no.copy_to(n_obs); d_psi.copy_to(psi); d_phi.copy_to(phi); d_nu.copy_to(nu);
    d_al.copy_to(alpha);
    return rc;
}

int simt_eval_trajectories(const float* psiphi, const double* times, int N, int H, int W, const int32_t* x0y0,
                           const float* vxvy, int M, float* Psi, float* Phi, int32_t* n_obs, int32_t* ixiy) {
    prep(0, 1);
    simt::DevBuf d_pp(psiphi, (size_t)N * H * W * 8), d_xy(x0y0, (size_t)M * 8), d_v(vxvy, (size_t)M * 8);
    simt::DevBuf d_psi((size_t)M * 4), d_phi((size_t)M * 4), d_no((size_t)M * 4), d_ix((size_t)M * N * 8);
    const int rc = launch_eval_trajectories(d_pp.as<const float2>(), dt_of(times, N), N, H, W, d_xy.as<const int32_t>(),
                                            d_v.as<const float2>(), M, d_psi.as<float>(), d_phi.as<float>(),
                                            d_no.as<int32_t>(), ixiy ? d_ix.as<int32_t>() : nullptr, nullptr);
    d_psi.copy_to(Psi); d_phi.copy_to(Phi); d_no.copy_to(n_obs);
    if (ixiy) d_ix.copy_to(ixiy);
    return rc;
}

long long simt_search_direct_threshold(const float* psiphi, const double* times, int N, int H, int W, const float* vel,
                                       int V, int min_obs, float nu_min, int y_begin, int y_end, long long capacity,
                                       int32_t* x, int32_t* y, int32_t* vel_idx, int32_t* n_obs, float* psi, float* phi,
                                       float* nu, float* alpha, int order, unsigned seed) {
    prep(order, seed);
    const size_t npix = (size_t)N * H * W, nc = (size_t)capacity * 4;
    simt::DevBuf d_pp(psiphi, npix * 8), d_vel(vel, (size_t)V * 8), d_count(8);
    simt::DevBuf d_x(nc), d_y(nc), d_vi(nc), d_no(nc), d_psi(nc), d_phi(nc), d_nu(nc), d_al(nc);
    *d_count.as<unsigned long long>() = 0;
    kbmod_candidates out{d_x.as<int32_t>(), d_y.as<int32_t>(), d_vi.as<int32_t>(), d_no.as<int32_t>(), d_psi.as<float>(),
                         d_phi.as<float>(), d_nu.as<float>(), d_al.as<float>()};
    const int rc = launch_search_direct_threshold(d_pp.as<const float2>(), dt_of(times, N), N, H, W,
                                                  d_vel.as<const float2>(), V, min_obs, nu_min, y_begin, y_end, out,
                                                  (unsigned long long)capacity, d_count.as<unsigned long long>(), nullptr);
    if (rc) return rc;
    d_x.copy_to(x); d_y.copy_to(y); d_vi.copy_to(vel_idx); d_no.copy_to(n_obs); d_psi.copy_to(psi); d_phi.copy_to(phi);
    d_nu.copy_to(nu); d_al.copy_to(alpha);
    return (long long)*d_count.as<unsigned long long>();
}

int simt_filter_candidates(const float* psiphi, const double* times, int N, int H, int W, const int32_t* x0y0,
                           const float* vxvy, int M, float sigma, float q, float* psi, float* phi, int32_t* n_obs,
                           float* nu, float* alpha, uint64_t* keep, float* kalman, int order, unsigned seed) {
    prep(order, seed);
    simt::DevBuf d_pp(psiphi, (size_t)N * H * W * 8), d_xy(x0y0, (size_t)M * 8), d_v(vxvy, (size_t)M * 8);
    simt::DevBuf d_psi((size_t)M * 4), d_phi((size_t)M * 4), d_no((size_t)M * 4), d_nu((size_t)M * 4), d_al((size_t)M * 4);
    simt::DevBuf d_keep((size_t)M * 8), d_kal((size_t)M * 8);
    const int rc = launch_filter_candidates(d_pp.as<const float2>(), dt_of(times, N), N, H, W, d_xy.as<const int32_t>(),
                                            d_v.as<const float2>(), M, sigma, q, d_psi.as<float>(), d_phi.as<float>(),
                                            d_no.as<int32_t>(), d_nu.as<float>(), d_al.as<float>(),
                                            d_keep.as<unsigned long long>(), d_kal.as<float2>(), nullptr);
    d_psi.copy_to(psi); d_phi.copy_to(phi); d_no.copy_to(n_obs); d_nu.copy_to(nu); d_al.copy_to(alpha);
    d_keep.copy_to(keep); d_kal.copy_to(kalman);
    return rc;
}

int simt_coadd_stamps(const float* sci, const uint8_t* mask, const double* times, int N, int H, int W,
                      const int32_t* x0y0, const float* vxvy, const uint64_t* keep, int M, int R, float* stamps,
                      float* moments, int order, unsigned seed) {
    prep(order, seed);
    const size_t npix = (size_t)N * H * W, S = 2 * (size_t)R + 1;
    simt::DevBuf d_sci(sci, npix * 4), d_mask(mask ? (const void*)mask : (const void*)sci, mask ? npix : 0);
    simt::DevBuf d_xy(x0y0, (size_t)M * 8), d_v(vxvy, (size_t)M * 8);
    simt::DevBuf d_keep(keep ? (const void*)keep : (const void*)sci, keep ? (size_t)M * 8 : 0);
    simt::DevBuf d_st((size_t)M * S * S * 4), d_mo((size_t)M * 24);
    const int rc = launch_coadd_stamps(d_sci.as<const float>(), mask ? d_mask.as<const uint8_t>() : nullptr,
                                       dt_of(times, N), N, H, W, d_xy.as<const int32_t>(), d_v.as<const float2>(),
                                       keep ? d_keep.as<const unsigned long long>() : nullptr, M, R, d_st.as<float>(),
                                       d_mo.as<float>(), nullptr);
    d_st.copy_to(stamps); d_mo.copy_to(moments);
    return rc;
}

int simt_cluster_candidates(const int32_t* x0y0, const float* vxvy, const float* nu, int M, float eps_xy, float eps_v,
                            int min_samples, int32_t* label, uint8_t* rep, int* launches, int order, unsigned seed) {
    prep(order, seed);
    simt::DevBuf d_xy(x0y0, (size_t)M * 8), d_v(vxvy, (size_t)M * 8), d_nu(nu, (size_t)M * 4);
    simt::DevBuf d_lab((size_t)M * 4), d_rep((size_t)M), d_ws(cluster_workspace_bytes(M));
    const int rc = launch_cluster_candidates(d_xy.as<const int32_t>(), d_v.as<const float2>(), d_nu.as<const float>(), M,
                                             eps_xy, eps_v, min_samples, d_lab.as<int32_t>(), d_rep.as<uint8_t>(), d_ws.p,
                                             nullptr);
    d_lab.copy_to(label); d_rep.copy_to(rep);
    *launches = (int)simt::S().launches;
    return rc;
}

int simt_build_mask(const float* sci, const float* var, const uint8_t* mask_in, int N, int H, int W, float sigma_thr,
                    int grow, int min_images, float bright, uint8_t* mask_out, int order, unsigned seed) {
    prep(order, seed);
    const size_t npix = (size_t)N * H * W;
    simt::DevBuf d_sci(sci, npix * 4), d_var(var, npix * 4), d_out(npix);
    simt::DevBuf d_in(mask_in ? (const void*)mask_in : (const void*)sci, mask_in ? npix : 0);
    const int rc = launch_build_mask(d_sci.as<const float>(), d_var.as<const float>(),
                                     mask_in ? d_in.as<const uint8_t>() : nullptr, N, H, W, sigma_thr, grow, min_images,
                                     bright, d_out.as<uint8_t>(), nullptr);
    d_out.copy_to(mask_out);
    return rc;
}

}  // extern "C"
