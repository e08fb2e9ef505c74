// api.cu -- the C ABI of include/kbmod_b200.h: argument checks, host-side plans, dispatch.
//
// No process-wide state selects anything: the search kernel and its tuning knobs arrive in a
// kbmod_search_options argument, the host plan lives in a caller-owned kbmod_plan object.  The only
// global is the launch counter (statistics).
#include <algorithm>
#include <atomic>
#include <cmath>
#include <cstring>
#include <new>
#include <vector>

#include "common.cuh"
#include "search_staged.cuh"
#include "search_tiled.cuh"

namespace kbmod {
static std::atomic<unsigned long long> g_launches{0};
void note_launch(int n) { g_launches.fetch_add((unsigned long long)n, std::memory_order_relaxed); }

static inline size_t align_up(size_t v, size_t a) { return (v + a - 1) / a * a; }

static int make_dt(const double* times, int N, DtTable& t) {
    for (int i = 0; i < KBMOD_MAX_IMAGES; ++i) t.dt[i] = 0.0f;
    for (int i = 0; i < N; ++i) {
        if (!std::isfinite(times[i])) return KBMOD_ERR_ARG;
        t.dt[i] = (float)(times[i] - times[0]);     // differenced in double, rounded once
    }
    return KBMOD_OK;
}

static bool have_device() {
    int n = 0;
    return cudaGetDeviceCount(&n) == cudaSuccess && n > 0;
}

struct WorkspaceLayout {
    size_t status_off, vel_off, plan_off, enc_off, total;
};

static WorkspaceLayout workspace_layout(int N, int H, int W, int V, int K) {
    WorkspaceLayout l;
    size_t off = 0;
    l.status_off = off;
    off = align_up(off + sizeof(int), 256);
    l.vel_off = off;
    off = align_up(off + (size_t)V * sizeof(float2), 256);
    l.plan_off = off;
    off = align_up(off + std::max(staged_plan_bytes(N, V), tiled_plan_bytes(N, V, K)), 256);
    l.enc_off = off;
    off = align_up(off + staged_enc_bytes(N, H, W), 256);
    l.total = off;
    return l;
}

// options with every default resolved; KBMOD_ERR_ARG for values out of range
struct Options {
    int kernel = KBMOD_KERNEL_AUTO, tile_group_w = 0, staged_geom = 0;
};
static int read_options(const kbmod_search_options* o, Options& out) {
    out = Options();
    if (!o) return KBMOD_OK;
    if (o->struct_size != 0 && o->struct_size != (int32_t)sizeof(kbmod_search_options)) return KBMOD_ERR_ARG;
    if (o->kernel < KBMOD_KERNEL_AUTO || o->kernel > KBMOD_KERNEL_TILED_QUEUED) return KBMOD_ERR_ARG;
    if (o->tile_group_w < 0 || o->tile_group_w > 256) return KBMOD_ERR_ARG;
    if (o->staged_geom < 0 || o->staged_geom > 3) return KBMOD_ERR_ARG;
    out.kernel = o->kernel;
    out.tile_group_w = o->tile_group_w;
    out.staged_geom = o->staged_geom;
    return KBMOD_OK;
}

// shared checks of the grid-shaped arguments (before any launch)
static int check_grid(const double* times, int N, int H, int W, const float* vel_grid, int V, int K) {
    if (!times || !vel_grid) return KBMOD_ERR_NULL;
    if (N <= 0 || H <= 0 || W <= 0 || V <= 0) return KBMOD_ERR_SHAPE;
    if (N > KBMOD_MAX_IMAGES || K > KBMOD_MAX_K) return KBMOD_ERR_UNSUPPORTED;
    if (K < 1) return KBMOD_ERR_ARG;
    for (int j = 0; j < 2 * V; ++j)
        if (!std::isfinite(vel_grid[j])) return KBMOD_ERR_ARG;
    for (int i = 0; i < N; ++i)
        if (!std::isfinite(times[i])) return KBMOD_ERR_ARG;
    return KBMOD_OK;
}
// planes may be NULL only when nothing will be written (an empty band of start rows)
static int check_result(const kbmod_result* out, bool empty = false) {
    if (!out) return KBMOD_ERR_NULL;
    if (!empty && (!out->vel_idx || !out->n_obs || !out->psi || !out->phi || !out->nu || !out->alpha))
        return KBMOD_ERR_NULL;
    if (((uintptr_t)out->vel_idx | (uintptr_t)out->n_obs | (uintptr_t)out->psi | (uintptr_t)out->phi |
         (uintptr_t)out->nu | (uintptr_t)out->alpha) & 3)
        return KBMOD_ERR_ALIGN;
    return KBMOD_OK;
}
}  // namespace kbmod

// The host plan (opaque to the caller): everything kbmod_search derives from (times, velocity grid,
// shape, K, options) before it looks at a pixel.  Immutable after kbmod_plan_create, so any number of
// searches on any streams may share it.
struct kbmod_plan {
    int N, H, W, V, K;
    int kernel;                   // resolved: never KBMOD_KERNEL_AUTO
    int tile_group_w;
    kbmod::DtTable dt;
    std::vector<float> vel;       // [V][2]
    kbmod::TiledPlan tiled;       // kernels 2 and 4
    kbmod::StagedPlan staged;     // kernel 3
};

using namespace kbmod;

extern "C" {

int kbmod_make_psi_phi(const float* sci, const float* var, const uint8_t* mask, const float* psf,
                       int N, int H, int W, int P, float* psiphi, void* stream) {
    if (!sci || !var || !psf || !psiphi) return KBMOD_ERR_NULL;
    if (N <= 0 || H <= 0 || W <= 0) return KBMOD_ERR_SHAPE;
    if (P <= 0 || (P % 2) == 0) return KBMOD_ERR_ARG;
    if (P > KBMOD_MAX_PSF) return KBMOD_ERR_UNSUPPORTED;
    if (((uintptr_t)psiphi & 7) || ((uintptr_t)sci & 3) || ((uintptr_t)var & 3)) return KBMOD_ERR_ALIGN;
    for (size_t k = 0; k < (size_t)N * P * P; ++k)
        if (!std::isfinite(psf[k])) return KBMOD_ERR_ARG;
    if (!have_device()) return KBMOD_ERR_CUDA;
    return launch_psi_phi(sci, var, mask, psf, N, H, W, P, reinterpret_cast<float2*>(psiphi),
                          (cudaStream_t)stream);
}

size_t kbmod_search_workspace(int N, int H, int W, int V, int K) {
    if (N <= 0 || H <= 0 || W <= 0 || V <= 0 || K <= 0) return 0;
    return workspace_layout(N, H, W, V, K).total;
}

int kbmod_plan_create(const double* times, int N, int H, int W, const float* vel_grid, int V, int K,
                      const kbmod_search_options* options, kbmod_plan** plan) {
    if (!plan) return KBMOD_ERR_NULL;
    *plan = nullptr;
    if (int rc = check_grid(times, N, H, W, vel_grid, V, K)) return rc;
    Options opt;
    if (int rc = read_options(options, opt)) return rc;
    kbmod_plan* p = new (std::nothrow) kbmod_plan();
    if (!p) return KBMOD_ERR_CUDA;
    p->N = N; p->H = H; p->W = W; p->V = V; p->K = K;
    p->tile_group_w = opt.tile_group_w;
    make_dt(times, N, p->dt);
    p->vel.assign(vel_grid, vel_grid + 2 * (size_t)V);
    int rc = KBMOD_OK;
    switch (opt.kernel) {
        case KBMOD_KERNEL_DIRECT:
            p->kernel = KBMOD_KERNEL_DIRECT;
            break;
        case KBMOD_KERNEL_STAGED:
            p->kernel = KBMOD_KERNEL_STAGED;
            rc = staged_plan_build(p->dt, N, H, W, vel_grid, V, opt.staged_geom, p->staged);
            break;
        case KBMOD_KERNEL_TILED:
        case KBMOD_KERNEL_TILED_QUEUED:
            p->kernel = opt.kernel;
            rc = tiled_plan_build(p->dt, N, H, W, vel_grid, V, K, opt.kernel == KBMOD_KERNEL_TILED_QUEUED, p->tiled);
            break;
        default:     // automatic: the tiled kernel where the shape fits, else the direct-gather kernel
            p->kernel = KBMOD_KERNEL_TILED;
            rc = tiled_plan_build(p->dt, N, H, W, vel_grid, V, K, false, p->tiled);
            if (rc == KBMOD_ERR_UNSUPPORTED) {
                p->kernel = KBMOD_KERNEL_DIRECT;
                rc = KBMOD_OK;
            }
            break;
    }
    if (rc != KBMOD_OK) {
        delete p;
        return rc;
    }
    *plan = p;
    return KBMOD_OK;
}

void kbmod_plan_destroy(kbmod_plan* plan) { delete plan; }

int kbmod_plan_kernel(const kbmod_plan* plan) { return plan ? plan->kernel : KBMOD_ERR_NULL; }

int kbmod_search_planned(const kbmod_plan* plan, const float* psiphi, int min_obs, int y_begin, int y_end,
                         const kbmod_result* out, void* workspace, size_t workspace_bytes, void* stream) {
    if (!plan || !psiphi || !workspace) return KBMOD_ERR_NULL;
    const int N = plan->N, H = plan->H, W = plan->W, V = plan->V, K = plan->K;
    if (min_obs < 1 || min_obs > N) return KBMOD_ERR_ARG;
    if (y_begin < 0 || y_end > H || y_begin > y_end) return KBMOD_ERR_ARG;
    if (int rc = check_result(out, y_begin == y_end)) return rc;
    if (((uintptr_t)psiphi & 15) || ((uintptr_t)workspace & 255)) return KBMOD_ERR_ALIGN;
    const WorkspaceLayout l = workspace_layout(N, H, W, V, K);
    if (workspace_bytes < l.total) return KBMOD_ERR_WORKSPACE;
    if (!have_device()) return KBMOD_ERR_CUDA;

    cudaStream_t st = (cudaStream_t)stream;
    char* ws = static_cast<char*>(workspace);
    const float2* pp = reinterpret_cast<const float2*>(psiphi);
    int* status_dev = reinterpret_cast<int*>(ws + l.status_off);
    if (cudaMemsetAsync(status_dev, 0, sizeof(int), st) != cudaSuccess) return KBMOD_ERR_CUDA;
    if (y_begin == y_end) return KBMOD_OK;                 // an empty band: nothing to search, nothing to write
    float2* vel_dev = reinterpret_cast<float2*>(ws + l.vel_off);
    if (cudaMemcpyAsync(vel_dev, plan->vel.data(), (size_t)V * sizeof(float2), cudaMemcpyHostToDevice, st) != cudaSuccess)
        return KBMOD_ERR_CUDA;
    float2* enc_dev = reinterpret_cast<float2*>(ws + l.enc_off);
    switch (plan->kernel) {
        case KBMOD_KERNEL_STAGED:
            return staged_launch(plan->staged, pp, plan->dt, N, H, W, K, min_obs, y_begin, y_end, *out,
                                 ws + l.plan_off, vel_dev, enc_dev, status_dev, st);
        case KBMOD_KERNEL_TILED:
        case KBMOD_KERNEL_TILED_QUEUED:
            return tiled_launch(plan->tiled, pp, plan->dt, N, H, W, K, min_obs, y_begin, y_end, *out,
                                ws + l.plan_off, vel_dev, enc_dev, plan->tile_group_w, st);
        default:
            return launch_search_direct(pp, plan->dt, N, H, W, vel_dev, V, K, min_obs, y_begin, y_end, *out, st);
    }
}

int kbmod_search_rows(const float* psiphi, const double* times, int N, int H, int W,
                      const float* vel_grid, int V, int K, int min_obs, int y_begin, int y_end,
                      const kbmod_result* out, void* workspace, size_t workspace_bytes,
                      const kbmod_search_options* options, void* stream) {
    // every argument error is found here, before the plan is built or anything is launched
    if (!psiphi || !workspace) return KBMOD_ERR_NULL;
    if (int rc = check_grid(times, N, H, W, vel_grid, V, K)) return rc;
    if (min_obs < 1 || min_obs > N) return KBMOD_ERR_ARG;
    if (y_begin < 0 || y_end > H || y_begin > y_end) return KBMOD_ERR_ARG;
    if (int rc = check_result(out, y_begin == y_end)) return rc;
    if (((uintptr_t)psiphi & 15) || ((uintptr_t)workspace & 255)) return KBMOD_ERR_ALIGN;
    if (workspace_bytes < workspace_layout(N, H, W, V, K).total) return KBMOD_ERR_WORKSPACE;
    Options opt;
    if (int rc = read_options(options, opt)) return rc;
    if (!have_device()) return KBMOD_ERR_CUDA;
    kbmod_plan* plan = nullptr;
    if (int rc = kbmod_plan_create(times, N, H, W, vel_grid, V, K, options, &plan)) return rc;
    const int rc = kbmod_search_planned(plan, psiphi, min_obs, y_begin, y_end, out, workspace, workspace_bytes, stream);
    kbmod_plan_destroy(plan);      // the launches have copied what they need (pageable copies are staged before return)
    return rc;
}

int kbmod_search(const float* psiphi, const double* times, int N, int H, int W,
                 const float* vel_grid, int V, int K, int min_obs, const kbmod_result* out,
                 void* workspace, size_t workspace_bytes, void* stream) {
    return kbmod_search_rows(psiphi, times, N, H, W, vel_grid, V, K, min_obs, 0, H, out, workspace,
                             workspace_bytes, nullptr, stream);
}

int kbmod_search_threshold(const float* psiphi, const double* times, int N, int H, int W,
                           const float* vel_grid, int V, int min_obs, float nu_min, int y_begin, int y_end,
                           const kbmod_candidates* out, long long capacity, unsigned long long* count,
                           void* workspace, size_t workspace_bytes, const kbmod_search_options* options,
                           void* stream) {
    if (!psiphi || !workspace || !out || !count) return KBMOD_ERR_NULL;
    if (capacity < 0) return KBMOD_ERR_ARG;
    if (capacity > 0 && (!out->x || !out->y || !out->vel_idx || !out->n_obs || !out->psi || !out->phi ||
                         !out->nu || !out->alpha))
        return KBMOD_ERR_NULL;
    constexpr int K = 8;                                   // sizes the plan and workspace of the tiled variant
    if (int rc = check_grid(times, N, H, W, vel_grid, V, K)) return rc;
    if (min_obs < 1 || min_obs > N) return KBMOD_ERR_ARG;
    if (!(nu_min == nu_min)) return KBMOD_ERR_ARG;         // NaN threshold
    if (y_begin < 0 || y_end > H || y_begin > y_end) return KBMOD_ERR_ARG;
    if (((uintptr_t)psiphi & 15) || ((uintptr_t)workspace & 255) || ((uintptr_t)count & 7)) return KBMOD_ERR_ALIGN;
    const WorkspaceLayout l = workspace_layout(N, H, W, V, K);
    if (workspace_bytes < l.total) return KBMOD_ERR_WORKSPACE;
    Options opt;
    if (int rc = read_options(options, opt)) return rc;
    if (opt.kernel == KBMOD_KERNEL_TILED || opt.kernel == KBMOD_KERNEL_STAGED) return KBMOD_ERR_UNSUPPORTED;
    DtTable dt;
    make_dt(times, N, dt);
    TiledPlan tplan;
    if (opt.kernel == KBMOD_KERNEL_TILED_QUEUED)
        if (int rc = tiled_plan_build(dt, N, H, W, vel_grid, V, K, true, tplan)) return rc;
    if (!have_device()) return KBMOD_ERR_CUDA;

    cudaStream_t st = (cudaStream_t)stream;
    char* ws = static_cast<char*>(workspace);
    const float2* pp = reinterpret_cast<const float2*>(psiphi);
    if (cudaMemsetAsync(ws + l.status_off, 0, sizeof(int), st) != cudaSuccess ||
        cudaMemsetAsync(count, 0, sizeof(unsigned long long), st) != cudaSuccess)
        return KBMOD_ERR_CUDA;
    float2* vel_dev = reinterpret_cast<float2*>(ws + l.vel_off);
    if (cudaMemcpyAsync(vel_dev, vel_grid, (size_t)V * sizeof(float2), cudaMemcpyHostToDevice, st) != cudaSuccess)
        return KBMOD_ERR_CUDA;
    if (opt.kernel == KBMOD_KERNEL_TILED_QUEUED)
        return tiled_launch_threshold(tplan, pp, dt, N, H, W, min_obs, nu_min, y_begin, y_end, *out,
                                      (unsigned long long)capacity, count, ws + l.plan_off, vel_dev,
                                      reinterpret_cast<float2*>(ws + l.enc_off), opt.tile_group_w, st);
    return launch_search_direct_threshold(pp, dt, N, H, W, vel_dev, V, min_obs, nu_min, y_begin, y_end, *out,
                                          (unsigned long long)capacity, count, st);
}

int kbmod_filter_candidates(const float* psiphi, const double* times, int N, int H, int W,
                            const int32_t* x0y0, const float* vxvy, int M, float sigma_reject,
                            float process_var, float* psi, float* phi, int32_t* n_obs, float* nu,
                            float* alpha, uint64_t* keep, float* kalman, void* stream) {
    if (!psiphi || !times || !psi || !phi || !n_obs || !nu || !alpha || !keep) return KBMOD_ERR_NULL;
    if (M > 0 && (!x0y0 || !vxvy)) return KBMOD_ERR_NULL;
    if (N <= 0 || H <= 0 || W <= 0 || M < 0) return KBMOD_ERR_SHAPE;
    if (N > KBMOD_MAX_IMAGES) return KBMOD_ERR_UNSUPPORTED;
    if (!(sigma_reject > 0.0f) || !std::isfinite(sigma_reject) || !(process_var >= 0.0f) || !std::isfinite(process_var))
        return KBMOD_ERR_ARG;
    if (((uintptr_t)psiphi & 7) || ((uintptr_t)vxvy & 7) || ((uintptr_t)keep & 7) || ((uintptr_t)kalman & 7))
        return KBMOD_ERR_ALIGN;
    DtTable dt;
    if (int rc = make_dt(times, N, dt)) return rc;
    if (!have_device()) return KBMOD_ERR_CUDA;
    return launch_filter_candidates(reinterpret_cast<const float2*>(psiphi), dt, N, H, W, x0y0,
                                    reinterpret_cast<const float2*>(vxvy), M, sigma_reject, process_var, psi, phi,
                                    n_obs, nu, alpha, reinterpret_cast<unsigned long long*>(keep),
                                    reinterpret_cast<float2*>(kalman), (cudaStream_t)stream);
}

int kbmod_coadd_stamps(const float* sci, const uint8_t* mask, const double* times, int N, int H, int W,
                       const int32_t* x0y0, const float* vxvy, const uint64_t* keep, int M, int R,
                       float* stamps, float* moments, void* stream) {
    if (!sci || !times || !stamps) return KBMOD_ERR_NULL;
    if (M > 0 && (!x0y0 || !vxvy)) return KBMOD_ERR_NULL;
    if (N <= 0 || H <= 0 || W <= 0 || M < 0) return KBMOD_ERR_SHAPE;
    if (R < 0) return KBMOD_ERR_ARG;
    if (N > KBMOD_MAX_IMAGES || R > 15) return KBMOD_ERR_UNSUPPORTED;
    if (((uintptr_t)sci & 3) || ((uintptr_t)vxvy & 7) || ((uintptr_t)keep & 7)) return KBMOD_ERR_ALIGN;
    DtTable dt;
    if (int rc = make_dt(times, N, dt)) return rc;
    if (!have_device()) return KBMOD_ERR_CUDA;
    return launch_coadd_stamps(sci, mask, dt, N, H, W, x0y0, reinterpret_cast<const float2*>(vxvy),
                               reinterpret_cast<const unsigned long long*>(keep), M, R, stamps, moments,
                               (cudaStream_t)stream);
}

int kbmod_build_mask(const float* sci, const float* var, const uint8_t* mask_in, int N, int H, int W,
                     float sigma_thr, int grow, int min_images, float bright_counts,
                     uint8_t* mask_out, void* stream) {
    if (!sci || !var || !mask_out) return KBMOD_ERR_NULL;
    if (N <= 0 || H <= 0 || W <= 0) return KBMOD_ERR_SHAPE;
    if (grow < 0 || min_images < 1 || !(sigma_thr == sigma_thr) || !(bright_counts == bright_counts)) return KBMOD_ERR_ARG;
    if (grow > 8) return KBMOD_ERR_UNSUPPORTED;
    if (((uintptr_t)sci & 3) || ((uintptr_t)var & 3)) return KBMOD_ERR_ALIGN;
    if (!have_device()) return KBMOD_ERR_CUDA;
    return launch_build_mask(sci, var, mask_in, N, H, W, sigma_thr, grow, min_images, bright_counts, mask_out,
                             (cudaStream_t)stream);
}

size_t kbmod_cluster_workspace(int M) { return M < 0 ? 0 : cluster_workspace_bytes(M); }

int kbmod_cluster_candidates(const int32_t* x0y0, const float* vxvy, const float* nu, int M,
                             float eps_xy, float eps_v, int min_samples, int32_t* label, uint8_t* rep,
                             void* workspace, size_t workspace_bytes, void* stream) {
    if (M < 0) return KBMOD_ERR_SHAPE;
    if (M > 0 && (!x0y0 || !vxvy || !nu || !label || !rep || !workspace)) return KBMOD_ERR_NULL;
    if (!(eps_xy > 0.0f) || !(eps_v > 0.0f) || !std::isfinite(eps_xy) || !std::isfinite(eps_v) || min_samples < 1)
        return KBMOD_ERR_ARG;
    if (((uintptr_t)vxvy & 7) || ((uintptr_t)workspace & 255)) return KBMOD_ERR_ALIGN;
    if (M > 0 && workspace_bytes < cluster_workspace_bytes(M)) return KBMOD_ERR_WORKSPACE;
    if (!have_device()) return KBMOD_ERR_CUDA;
    return launch_cluster_candidates(x0y0, reinterpret_cast<const float2*>(vxvy), nu, M, eps_xy, eps_v, min_samples,
                                     label, rep, workspace, (cudaStream_t)stream);
}

int kbmod_search_status(const void* workspace, void* stream) {
    if (!workspace) return KBMOD_ERR_NULL;
    if ((uintptr_t)workspace & 255) return KBMOD_ERR_ALIGN;
    if (!have_device()) return KBMOD_ERR_CUDA;
    int status = 0;
    if (cudaMemcpyAsync(&status, workspace, sizeof(int), cudaMemcpyDeviceToHost, (cudaStream_t)stream) != cudaSuccess ||
        cudaStreamSynchronize((cudaStream_t)stream) != cudaSuccess)
        return KBMOD_ERR_CUDA;
    return status == 0 ? KBMOD_OK : KBMOD_ERR_TIMEOUT;
}

namespace kbmod {
struct HostLayout {
    size_t search_off, sci_off, var_off, mask_off, pp_off, plane_off[6], total;
};
static HostLayout host_layout(int N, int H, int W, int V, int K) {
    HostLayout l;
    const size_t px = (size_t)N * H * W, rk = (size_t)H * W * K;
    size_t off = 0;
    l.search_off = off;                       // first: kbmod_search_status reads word 0 of the workspace
    off = align_up(off + workspace_layout(N, H, W, V, K).total, 256);
    l.sci_off = off; off = align_up(off + px * 4, 256);
    l.var_off = off; off = align_up(off + px * 4, 256);
    l.mask_off = off; off = align_up(off + px, 256);
    l.pp_off = off; off = align_up(off + px * 8, 256);
    for (int k = 0; k < 6; ++k) { l.plane_off[k] = off; off = align_up(off + rk * 4, 256); }
    l.total = off;
    return l;
}
}  // namespace kbmod

size_t kbmod_search_host_workspace(int N, int H, int W, int V, int K) {
    if (N <= 0 || H <= 0 || W <= 0 || V <= 0 || K <= 0) return 0;
    return host_layout(N, H, W, V, K).total;
}

int kbmod_search_host(const float* sci, const float* var, const uint8_t* mask, const float* psf,
                      const double* times, int N, int H, int W, int P, const float* vel_grid, int V,
                      int K, int min_obs, const kbmod_result* out, void* workspace,
                      size_t workspace_bytes, const kbmod_search_options* options, void* stream) {
    // every argument error of both stages is found here, before the first copy is enqueued
    if (!sci || !var || !psf || !workspace) return KBMOD_ERR_NULL;
    if (int rc = check_result(out)) return rc;
    if (int rc = check_grid(times, N, H, W, vel_grid, V, K)) return rc;
    if (min_obs < 1 || min_obs > N) return KBMOD_ERR_ARG;
    if (P <= 0 || (P % 2) == 0) return KBMOD_ERR_ARG;
    if (P > KBMOD_MAX_PSF) return KBMOD_ERR_UNSUPPORTED;
    for (size_t k = 0; k < (size_t)N * P * P; ++k)
        if (!std::isfinite(psf[k])) return KBMOD_ERR_ARG;
    if (((uintptr_t)workspace & 255) || ((uintptr_t)sci & 3) || ((uintptr_t)var & 3)) return KBMOD_ERR_ALIGN;
    Options opt;
    if (int rc = read_options(options, opt)) return rc;
    const HostLayout l = host_layout(N, H, W, V, K);
    if (workspace_bytes < l.total) return KBMOD_ERR_WORKSPACE;
    if (!have_device()) return KBMOD_ERR_CUDA;
    kbmod_plan* plan = nullptr;
    if (int rc = kbmod_plan_create(times, N, H, W, vel_grid, V, K, options, &plan)) return rc;

    cudaStream_t st = (cudaStream_t)stream;
    char* ws = static_cast<char*>(workspace);
    const size_t px = (size_t)N * H * W, rk = (size_t)H * W * K;
    float* d_sci = reinterpret_cast<float*>(ws + l.sci_off);
    float* d_var = reinterpret_cast<float*>(ws + l.var_off);
    uint8_t* d_mask = mask ? reinterpret_cast<uint8_t*>(ws + l.mask_off) : nullptr;
    float* d_pp = reinterpret_cast<float*>(ws + l.pp_off);
    int rc = KBMOD_OK;
    if (cudaMemcpyAsync(d_sci, sci, px * 4, cudaMemcpyHostToDevice, st) != cudaSuccess ||
        cudaMemcpyAsync(d_var, var, px * 4, cudaMemcpyHostToDevice, st) != cudaSuccess ||
        (mask && cudaMemcpyAsync(d_mask, mask, px, cudaMemcpyHostToDevice, st) != cudaSuccess))
        rc = KBMOD_ERR_CUDA;
    if (rc == KBMOD_OK) rc = kbmod_make_psi_phi(d_sci, d_var, d_mask, psf, N, H, W, P, d_pp, stream);
    kbmod_result dev;
    void* host_planes[6] = {out->vel_idx, out->n_obs, out->psi, out->phi, out->nu, out->alpha};
    void* dev_planes[6];
    for (int k = 0; k < 6; ++k) dev_planes[k] = ws + l.plane_off[k];
    dev.vel_idx = static_cast<int32_t*>(dev_planes[0]);
    dev.n_obs = static_cast<int32_t*>(dev_planes[1]);
    dev.psi = static_cast<float*>(dev_planes[2]);
    dev.phi = static_cast<float*>(dev_planes[3]);
    dev.nu = static_cast<float*>(dev_planes[4]);
    dev.alpha = static_cast<float*>(dev_planes[5]);
    if (rc == KBMOD_OK)
        rc = kbmod_search_planned(plan, d_pp, min_obs, 0, H, &dev, ws + l.search_off,
                                  workspace_layout(N, H, W, V, K).total, stream);
    kbmod_plan_destroy(plan);
    if (rc != KBMOD_OK) return rc;
    for (int k = 0; k < 6; ++k)
        if (cudaMemcpyAsync(host_planes[k], dev_planes[k], rk * 4, cudaMemcpyDeviceToHost, st) != cudaSuccess)
            return KBMOD_ERR_CUDA;
    return KBMOD_OK;
}

int kbmod_search_split(const float* psi, const float* phi, const double* times, int N, int H,
                       int W, const float* vel_grid, int V, int K, int min_obs,
                       const kbmod_result* out, void* workspace, size_t workspace_bytes,
                       void* stream) {
    if (!psi || !phi || !workspace) return KBMOD_ERR_NULL;
    if (int rc = check_result(out)) return rc;
    if (int rc = check_grid(times, N, H, W, vel_grid, V, K)) return rc;
    if (min_obs < 1 || min_obs > N) return KBMOD_ERR_ARG;
    if ((uintptr_t)workspace & 255) return KBMOD_ERR_ALIGN;
    const size_t need = kbmod_search_workspace(N, H, W, V, K);
    const size_t n = (size_t)N * H * W;
    if (workspace_bytes < need + n * sizeof(float2)) return KBMOD_ERR_WORKSPACE;
    if (!have_device()) return KBMOD_ERR_CUDA;
    float2* inter = reinterpret_cast<float2*>(static_cast<char*>(workspace) + need);
    if (int rc = launch_interleave(psi, phi, n, inter, (cudaStream_t)stream)) return rc;
    return kbmod_search(reinterpret_cast<const float*>(inter), times, N, H, W, vel_grid, V, K,
                        min_obs, out, workspace, need, stream);
}

int kbmod_eval_trajectories(const float* psiphi, const double* times, int N, int H, int W,
                            const int32_t* x0y0, const float* vxvy, int M, float* Psi, float* Phi,
                            int32_t* n_obs, int32_t* ixiy, void* stream) {
    if (!psiphi || !times || !Psi || !Phi || !n_obs) return KBMOD_ERR_NULL;
    if (M > 0 && (!x0y0 || !vxvy)) return KBMOD_ERR_NULL;
    if (N <= 0 || H <= 0 || W <= 0 || M < 0) return KBMOD_ERR_SHAPE;
    if (N > KBMOD_MAX_IMAGES) return KBMOD_ERR_UNSUPPORTED;
    if (((uintptr_t)psiphi & 7) || ((uintptr_t)vxvy & 7)) return KBMOD_ERR_ALIGN;
    DtTable dt;
    if (int rc = make_dt(times, N, dt)) return rc;
    if (!have_device()) return KBMOD_ERR_CUDA;
    return launch_eval_trajectories(reinterpret_cast<const float2*>(psiphi), dt, N, H, W, x0y0,
                                    reinterpret_cast<const float2*>(vxvy), M, Psi, Phi, n_obs, ixiy,
                                    (cudaStream_t)stream);
}

int kbmod_debug_staged_plan(const double* times, int N, int H, int W, const float* vel_grid, int V,
                            int staged_geom, int32_t* stream, size_t stream_ints, int32_t* shapes,
                            int max_shapes, int32_t* info) {
    if (!times || !vel_grid || !stream || !shapes || !info) return KBMOD_ERR_NULL;
    if (N <= 0 || H <= 0 || W <= 0 || V <= 0 || max_shapes < 0) return KBMOD_ERR_SHAPE;
    if (N > KBMOD_MAX_IMAGES) return KBMOD_ERR_UNSUPPORTED;
    for (int j = 0; j < 2 * V; ++j)
        if (!std::isfinite(vel_grid[j])) return KBMOD_ERR_ARG;
    DtTable dt;
    if (int rc = make_dt(times, N, dt)) return rc;
    return staged_plan_debug(dt, N, H, W, vel_grid, V, staged_geom, stream, stream_ints, shapes, max_shapes, info);
}

unsigned long long kbmod_launch_count(void) { return g_launches.load(); }

const char* kbmod_status_string(int status) {
    switch (status) {
        case KBMOD_OK: return "ok";
        case KBMOD_ERR_NULL: return "required pointer is NULL";
        case KBMOD_ERR_SHAPE: return "non-positive or inconsistent dimension";
        case KBMOD_ERR_ARG: return "argument out of range";
        case KBMOD_ERR_ALIGN: return "pointer not aligned as documented";
        case KBMOD_ERR_CUDA: return "CUDA error or no CUDA device";
        case KBMOD_ERR_UNSUPPORTED: return "beyond the supported limits";
        case KBMOD_ERR_WORKSPACE: return "workspace too small";
        case KBMOD_ERR_TIMEOUT: return "a kernel gave up waiting on its own pipeline";
    }
    return "unknown status";
}

const char* kbmod_version(void) { return "0.2"; }

}  // extern "C"
