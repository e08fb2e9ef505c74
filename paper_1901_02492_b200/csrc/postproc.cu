// postproc.cu -- the rows around the search: N1 light-curve outlier
// filter and re-score, N2 coadded postage stamps and central moments, N3 mask builder.
//
// These are small, regular kernels (candidates number 1e5..1e6, "70 seconds for 500,000
// objects" in the paper's Python): one thread or one CTA per candidate, literal S3 (traj_pixel) for
// every sampled position.  Every floating-point DECISION (outlier or not, detected or not) is taken
// with separately rounded binary32 operations in a fixed order, which the oracle restates, so the
// integer outputs are bit-exact; the readings of what the paper leaves open are DESIGN.md's
// N1-a..e, N2-a..c, N3-a..c.
#include "common.cuh"

namespace kbmod {

namespace {
__device__ __forceinline__ bool finitef(float v) { return fabsf(v) <= 3.402823466e38f; }
}  // namespace

// ---------------------------------------------------------------------------------------------
// N1  (section 3.3)
// ---------------------------------------------------------------------------------------------
struct KalmanPass {
    int n_kept;
    unsigned long long keep;
    float x, P;
};

// One pass of the scalar Kalman filter over the usable observations, forward or backward.
__device__ __forceinline__ KalmanPass kalman_pass(const float* psi, const float* phi, unsigned long long usable,
                                                  int N, bool backward, float q, float s2) {
    KalmanPass o{0, 0ull, 0.0f, 0.0f};
    bool have = false;
    float x = 0.0f, P = 0.0f;
    for (int k = 0; k < N; ++k) {
        const int i = backward ? N - 1 - k : k;
        if (!((usable >> i) & 1ull)) continue;
        const float f = __fdiv_rn(psi[i], phi[i]);       // flux of the observation (Eq.22)
        const float r = __fdiv_rn(1.0f, phi[i]);         // its variance
        if (!have) {
            x = f; P = r; have = true;
            o.keep |= 1ull << i; ++o.n_kept;
            continue;
        }
        const float Pp = __fadd_rn(P, q);
        const float e = __fsub_rn(f, x);
        const float S = __fadd_rn(Pp, r);
        if (__fmul_rn(e, e) > __fmul_rn(s2, S)) {
            P = Pp;                                      // outlier: not ingested
        } else {
            const float G = __fdiv_rn(Pp, S);
            x = __fadd_rn(x, __fmul_rn(G, e));
            P = __fmul_rn(__fsub_rn(1.0f, G), Pp);
            o.keep |= 1ull << i; ++o.n_kept;
        }
    }
    o.x = x; o.P = P;
    return o;
}

__global__ void __launch_bounds__(128)
filter_candidates_kernel(const float2* __restrict__ psiphi, const __grid_constant__ DtTable dt, int N, int H, int W,
                         const int32_t* __restrict__ x0y0, const float2* __restrict__ vxvy, int M, float s2, float q,
                         float* o_psi, float* o_phi, int32_t* o_nobs, float* o_nu, float* o_alpha,
                         unsigned long long* o_keep, float2* o_kalman) {
    const int m = blockIdx.x * blockDim.x + threadIdx.x;
    if (m >= M) return;
    float psi[KBMOD_MAX_IMAGES], phi[KBMOD_MAX_IMAGES];
    unsigned long long exists = 0ull, usable = 0ull;
    const int x0 = x0y0[2 * m], y0 = x0y0[2 * m + 1];
    const float2 v = vxvy[m];
    for (int i = 0; i < N; ++i) {
        int ix, iy;
        psi[i] = 0.0f; phi[i] = 0.0f;
        if (traj_pixel(x0, v.x, dt.dt[i], W, ix) && traj_pixel(y0, v.y, dt.dt[i], H, iy)) {
            const float2 s = __ldg(psiphi + ((size_t)i * H + iy) * W + ix);
            if (s.x == s.x) {
                psi[i] = s.x; phi[i] = s.y;
                exists |= 1ull << i;
                if (s.y > 0.0f) usable |= 1ull << i;
            }
        }
    }
    const KalmanPass fw = kalman_pass(psi, phi, usable, N, false, q, s2);
    const KalmanPass bw = kalman_pass(psi, phi, usable, N, true, q, s2);
    const bool take_bw = bw.n_kept > fw.n_kept;          // the pass that keeps more decides; tie: forward
    const unsigned long long keep = (exists & ~usable) | (take_bw ? bw.keep : fw.keep);
    float Psi = 0.0f, Phi = 0.0f;
    int n = 0;
    for (int i = 0; i < N; ++i)
        if ((keep >> i) & 1ull) {
            Psi = __fadd_rn(Psi, psi[i]);
            Phi = __fadd_rn(Phi, phi[i]);
            ++n;
        }
    const bool ok = n > 0 && Phi > 0.0f;
    o_psi[m] = Psi; o_phi[m] = Phi; o_nobs[m] = n; o_keep[m] = keep;
    o_nu[m] = ok ? score_nu(Psi, Phi) : -INFINITY;
    o_alpha[m] = ok ? score_alpha(Psi, Phi) : 0.0f;
    if (o_kalman) o_kalman[m] = take_bw ? make_float2(bw.x, bw.P) : make_float2(fw.x, fw.P);
}

int launch_filter_candidates(const float2* psiphi, const DtTable& dt, int N, int H, int W, const int32_t* x0y0,
                             const float2* vxvy, int M, float sigma_reject, float q, float* psi, float* phi,
                             int32_t* n_obs, float* nu, float* alpha, unsigned long long* keep, float2* kalman,
                             cudaStream_t st) {
    if (M == 0) return KBMOD_OK;
    volatile float s2 = sigma_reject * sigma_reject;     // one binary32 multiply
    KBMOD_LAUNCH(filter_candidates_kernel, (M + 127) / 128, 128, 0, st, psiphi, dt, N, H, W, x0y0, vxvy, M,
                 (float)s2, q, psi, phi, n_obs, nu, alpha, keep, kalman);
    note_launch();
    return cudaGetLastError() == cudaSuccess ? KBMOD_OK : KBMOD_ERR_CUDA;
}

// ---------------------------------------------------------------------------------------------
// N2  (section 3.3)
// ---------------------------------------------------------------------------------------------
constexpr int STAMP_THREADS = 128;
constexpr int STAMP_MAX_R = 15;                          // 31 x 31 pixels

// One CTA per candidate.  Pixels of the stamp in parallel (each a mean over the contributing
// images, image order); then one thread accumulates the moments row-major, as the definition does.
__global__ void __launch_bounds__(STAMP_THREADS)
coadd_stamps_kernel(const float* __restrict__ sci, const uint8_t* __restrict__ mask,
                    const __grid_constant__ DtTable dt, int N, int H, int W, const int32_t* __restrict__ x0y0,
                    const float2* __restrict__ vxvy, const unsigned long long* __restrict__ keep, int M, int R,
                    float* __restrict__ stamps, float* __restrict__ moments) {
    extern __shared__ __align__(16) unsigned char smem_raw[];     // ix[64], iy[64], stamp[S*S]
    int* s_ix = reinterpret_cast<int*>(smem_raw);
    int* s_iy = s_ix + KBMOD_MAX_IMAGES;
    float* s_st = reinterpret_cast<float*>(s_iy + KBMOD_MAX_IMAGES);
    const int m = blockIdx.x, tid = threadIdx.x;
    const int S = 2 * R + 1;
    if (tid < N) {
        const float2 v = vxvy[m];
        int ix = 0, iy = 0;
        const bool on = traj_pixel(x0y0[2 * m], v.x, dt.dt[tid], W, ix) &&
                        traj_pixel(x0y0[2 * m + 1], v.y, dt.dt[tid], H, iy) &&
                        (!keep || ((keep[m] >> tid) & 1ull));
        s_ix[tid] = on ? ix : -1;
        s_iy[tid] = iy;
    }
    __syncthreads();
    for (int p = tid; p < S * S; p += STAMP_THREADS) {
        const int dy = p / S - R, dx = p - (p / S) * S - R;
        float sum = 0.0f;
        int n = 0;
        for (int i = 0; i < N; ++i) {
            if (s_ix[i] < 0) continue;
            const int yy = s_iy[i] + dy, xx = s_ix[i] + dx;
            if (yy < 0 || yy >= H || xx < 0 || xx >= W) continue;
            const size_t k = ((size_t)i * H + yy) * W + xx;
            if (mask && __ldg(mask + k)) continue;
            const float v = __ldg(sci + k);
            if (!finitef(v)) continue;
            sum = __fadd_rn(sum, v);
            ++n;
        }
        const float mean = n ? __fdiv_rn(sum, (float)n) : 0.0f;
        s_st[p] = mean;
        stamps[(size_t)m * S * S + p] = mean;
    }
    __syncthreads();
    if (tid != 0 || !moments) return;
    float* mo = moments + (size_t)m * 6;
    float m00 = 0.0f, sx = 0.0f, sy = 0.0f;
    for (int dy = -R; dy <= R; ++dy)
        for (int dx = -R; dx <= R; ++dx) {
            const float w = fmaxf(s_st[(dy + R) * S + (dx + R)], 0.0f);
            m00 = __fadd_rn(m00, w);
            sx = __fadd_rn(sx, __fmul_rn(w, (float)dx));
            sy = __fadd_rn(sy, __fmul_rn(w, (float)dy));
        }
    if (!(m00 > 0.0f)) {
        for (int k = 0; k < 6; ++k) mo[k] = 0.0f;
        return;
    }
    const float cx = __fdiv_rn(sx, m00), cy = __fdiv_rn(sy, m00);
    float s20 = 0.0f, s02 = 0.0f, s11 = 0.0f;
    for (int dy = -R; dy <= R; ++dy)
        for (int dx = -R; dx <= R; ++dx) {
            const float w = fmaxf(s_st[(dy + R) * S + (dx + R)], 0.0f);
            const float ux = __fsub_rn((float)dx, cx), uy = __fsub_rn((float)dy, cy);
            const float wux = __fmul_rn(w, ux), wuy = __fmul_rn(w, uy);
            s20 = __fadd_rn(s20, __fmul_rn(wux, ux));
            s02 = __fadd_rn(s02, __fmul_rn(wuy, uy));
            s11 = __fadd_rn(s11, __fmul_rn(wux, uy));
        }
    mo[0] = m00; mo[1] = cx; mo[2] = cy;
    mo[3] = __fdiv_rn(s20, m00); mo[4] = __fdiv_rn(s02, m00); mo[5] = __fdiv_rn(s11, m00);
}

int launch_coadd_stamps(const float* sci, const uint8_t* mask, const DtTable& dt, int N, int H, int W,
                        const int32_t* x0y0, const float2* vxvy, const unsigned long long* keep, int M, int R,
                        float* stamps, float* moments, cudaStream_t st) {
    if (R < 0 || R > STAMP_MAX_R) return KBMOD_ERR_UNSUPPORTED;
    if (M == 0) return KBMOD_OK;
    const size_t smem = 2 * KBMOD_MAX_IMAGES * sizeof(int) + (size_t)(2 * R + 1) * (2 * R + 1) * sizeof(float);
    KBMOD_LAUNCH(coadd_stamps_kernel, M, STAMP_THREADS, smem, st, sci, mask, dt, N, H, W, x0y0, vxvy, keep, M, R,
                 stamps, moments);
    note_launch();
    return cudaGetLastError() == cudaSuccess ? KBMOD_OK : KBMOD_ERR_CUDA;
}

// ---------------------------------------------------------------------------------------------
// N3  (section 3.2; section 5.2)
// ---------------------------------------------------------------------------------------------
constexpr int MASK_TILE = 32;                            // 32 x 32 output pixels per CTA, 1024 threads
constexpr int MASK_MAX_GROW = 8;

// One CTA per tile; it walks the N images twice.  Pass 1: the detection map of tile + halo of image i
// is staged in shared memory, every thread ORs the disc around its pixel and counts the images in
// which the grown detection covers it.  Pass 2: mask_i = mask_in_i | static | bright_i.
__global__ void __launch_bounds__(MASK_TILE * MASK_TILE)
build_mask_kernel(const float* __restrict__ sci, const float* __restrict__ var, const uint8_t* __restrict__ mask_in,
                  int N, int H, int W, int tiles_x, float sigma_thr, int grow, int min_images, float bright_counts,
                  uint8_t* __restrict__ mask_out) {
    constexpr int SW = MASK_TILE + 2 * MASK_MAX_GROW;
    extern __shared__ __align__(16) unsigned char smem_raw[];     // detection map of tile + halo: SW x SW bytes
    uint8_t* s_det = smem_raw;
    const int tx = threadIdx.x & (MASK_TILE - 1), ty = threadIdx.x / MASK_TILE;
    const int x_tile = (blockIdx.x % tiles_x) * MASK_TILE, y_tile = (blockIdx.x / tiles_x) * MASK_TILE;
    const int x = x_tile + tx, y = y_tile + ty;
    const int sw = MASK_TILE + 2 * grow;
    const size_t npx = (size_t)H * W;
    int cnt = 0;
    for (int i = 0; i < N; ++i) {
        __syncthreads();
        for (int k = threadIdx.x; k < sw * sw; k += MASK_TILE * MASK_TILE) {
            const int sy = k / sw, sx = k - sy * sw;
            const int gy = y_tile + sy - grow, gx = x_tile + sx - grow;
            uint8_t d = 0;
            if (gy >= 0 && gy < H && gx >= 0 && gx < W) {
                const float s = __ldg(sci + i * npx + (size_t)gy * W + gx);
                const float v = __ldg(var + i * npx + (size_t)gy * W + gx);
                if (finitef(s) && finitef(v) && v > 0.0f) d = s > __fmul_rn(sigma_thr, __fsqrt_rn(v));
            }
            s_det[sy * SW + sx] = d;
        }
        __syncthreads();
        int g = 0;
        for (int dy = -grow; dy <= grow; ++dy)
            for (int dx = -grow; dx <= grow; ++dx)
                if (dx * dx + dy * dy <= grow * grow) g |= s_det[(ty + grow + dy) * SW + (tx + grow + dx)];
        cnt += g;
    }
    if (x >= W || y >= H) return;
    const bool is_static = cnt >= min_images;
    for (int i = 0; i < N; ++i) {
        const size_t k = i * npx + (size_t)y * W + x;
        const float s = __ldg(sci + k);
        bool m = mask_in ? (__ldg(mask_in + k) != 0) : false;
        m = m || is_static || (finitef(s) && s > bright_counts);
        mask_out[k] = m ? 1 : 0;
    }
}

int launch_build_mask(const float* sci, const float* var, const uint8_t* mask_in, int N, int H, int W,
                      float sigma_thr, int grow, int min_images, float bright_counts, uint8_t* mask_out,
                      cudaStream_t st) {
    if (grow > MASK_MAX_GROW) return KBMOD_ERR_UNSUPPORTED;
    const long long gx = (W + MASK_TILE - 1) / MASK_TILE, gy = (H + MASK_TILE - 1) / MASK_TILE;
    if (gx * gy > 0x7FFFFFFFLL) return KBMOD_ERR_UNSUPPORTED;
    constexpr int SW = MASK_TILE + 2 * MASK_MAX_GROW;
    KBMOD_LAUNCH(build_mask_kernel, (unsigned)(gx * gy), MASK_TILE * MASK_TILE, SW * SW, st, sci, var, mask_in, N, H, W,
                 (int)gx, sigma_thr, grow, min_images, bright_counts, mask_out);
    note_launch();
    return cudaGetLastError() == cudaSuccess ? KBMOD_OK : KBMOD_ERR_CUDA;
}

}  // namespace kbmod

// ---------------------------------------------------------------------------------------------
// N5  (section 3.3): DBSCAN over (x0, y0, vx, vy), brightest member per cluster
// ---------------------------------------------------------------------------------------------
// Candidate lists are short (the paper's filters leave 1e2..1e5 per field), so all-pairs passes are
// the simple and regular choice: every kernel below walks the M points in shared-memory tiles.
// The neighbour test is the fixed binary32 sequence DESIGN.md N5-a states; labels are canonical
// (smallest core index of the component), found by min-label propagation with pointer jumping.
namespace kbmod {

constexpr int CL_THREADS = 256;
constexpr int CL_NOLABEL = 0x7FFFFFFF;

struct ClPoint { int x, y; float vx, vy; };

__device__ __forceinline__ bool cl_neighbours(const ClPoint& a, const ClPoint& b, float ixy, float iv) {
    const long long dx = (long long)a.x - b.x, dy = (long long)a.y - b.y;
    const float r2 = (float)(dx * dx + dy * dy);
    const float dvx = __fsub_rn(a.vx, b.vx), dvy = __fsub_rn(a.vy, b.vy);
    const float v2 = __fadd_rn(__fmul_rn(dvx, dvx), __fmul_rn(dvy, dvy));
    return __fadd_rn(__fmul_rn(r2, ixy), __fmul_rn(v2, iv)) <= 1.0f;
}

__device__ __forceinline__ ClPoint cl_load(const int32_t* x0y0, const float2* vxvy, int i) {
    const float2 v = vxvy[i];
    return ClPoint{x0y0[2 * i], x0y0[2 * i + 1], v.x, v.y};
}

// mode 0: core[i] = (#neighbours >= min_samples), label[i] = core ? i : NOLABEL
// mode 1: one propagation step over core points: label[i] = min(label[i], labels of core neighbours); *changed |= moved
// mode 2: border / noise: non-core i takes the smallest label among its core neighbours, else -1
// mode 3: rep[i] = no member of the same cluster ranks before i (larger nu; equal nu: smaller index); noise: 1
__global__ void __launch_bounds__(CL_THREADS)
cluster_pass_kernel(int mode, const int32_t* __restrict__ x0y0, const float2* __restrict__ vxvy,
                    const float* __restrict__ nu, int M, float ixy, float iv, int min_samples, uint8_t* core,
                    const int32_t* label_in, int32_t* label_out, uint8_t* rep, int* changed) {
    extern __shared__ __align__(16) unsigned char smem_raw[];
    ClPoint* s_pt = reinterpret_cast<ClPoint*>(smem_raw);                       // [CL_THREADS]
    int* s_lab = reinterpret_cast<int*>(s_pt + CL_THREADS);                     // label (or core flag in mode 0)
    float* s_nu = reinterpret_cast<float*>(s_lab + CL_THREADS);
    unsigned char* s_core = reinterpret_cast<unsigned char*>(s_nu + CL_THREADS);
    const int i = blockIdx.x * CL_THREADS + threadIdx.x;
    const bool live = i < M;
    const ClPoint me = live ? cl_load(x0y0, vxvy, i) : ClPoint{0, 0, 0.0f, 0.0f};
    const int my_lab = (live && mode != 0) ? label_in[i] : CL_NOLABEL;
    const bool my_core = (live && mode != 0) ? core[i] != 0 : false;
    const float my_nu = (live && mode == 3) ? nu[i] : 0.0f;
    int count = 0, best = CL_NOLABEL;
    bool beaten = false;
    for (int j0 = 0; j0 < M; j0 += CL_THREADS) {
        __syncthreads();
        const int j = j0 + threadIdx.x;
        if (j < M) {
            s_pt[threadIdx.x] = cl_load(x0y0, vxvy, j);
            s_lab[threadIdx.x] = mode != 0 ? label_in[j] : 0;
            s_core[threadIdx.x] = mode != 0 ? core[j] : 0;
            s_nu[threadIdx.x] = mode == 3 ? nu[j] : 0.0f;
        }
        __syncthreads();
        const int n = min(CL_THREADS, M - j0);
        if (!live) continue;
        for (int k = 0; k < n; ++k) {
            if (mode == 3) {
                if (my_lab >= 0 && s_lab[k] == my_lab && j0 + k != i &&
                    (s_nu[k] > my_nu || (s_nu[k] == my_nu && j0 + k < i)))
                    beaten = true;
                continue;
            }
            if (mode != 0 && !s_core[k]) continue;
            if (!cl_neighbours(me, s_pt[k], ixy, iv)) continue;
            ++count;
            best = min(best, s_lab[k]);
        }
    }
    if (!live) return;
    if (mode == 0) {
        const bool c = count >= min_samples;
        core[i] = c;
        label_out[i] = c ? i : CL_NOLABEL;
    } else if (mode == 1) {
        int l = my_lab;
        if (my_core && best < l) { l = best; *changed = 1; }
        label_out[i] = l;
    } else if (mode == 2) {
        label_out[i] = my_core ? my_lab : (best == CL_NOLABEL ? -1 : best);
    } else {
        rep[i] = (my_lab < 0 || !beaten) ? 1 : 0;
    }
}

// pointer jumping between propagation steps: a core point's label is a core index of its own
// component (or its own), so label[label[i]] is a smaller-or-equal index of the same component
__global__ void __launch_bounds__(CL_THREADS)
cluster_jump_kernel(const uint8_t* __restrict__ core, const int32_t* label_in, int32_t* label_out, int M) {
    const int i = blockIdx.x * CL_THREADS + threadIdx.x;
    if (i >= M) return;
    int l = label_in[i];
    if (core[i]) {
        const int l2 = label_in[l];
        if (l2 < l) l = l2;
    }
    label_out[i] = l;
}

size_t cluster_workspace_bytes(int M) {
    const size_t m = (size_t)(M > 0 ? M : 1);
    return ((m + 255) / 256 * 256) + 2 * ((m * 4 + 255) / 256 * 256) + 256;      // core, two label buffers, flag
}

// SYNCHRONISES the stream once per propagation round (the number of rounds depends on the data).
int launch_cluster_candidates(const int32_t* x0y0, const float2* vxvy, const float* nu, int M, float eps_xy,
                              float eps_v, int min_samples, int32_t* label, uint8_t* rep, void* workspace,
                              cudaStream_t st) {
    if (M == 0) return KBMOD_OK;
    volatile float exy2 = eps_xy * eps_xy, ev2 = eps_v * eps_v;
    volatile float ixy = 1.0f / exy2, iv = 1.0f / ev2;
    char* ws = static_cast<char*>(workspace);
    const size_t mb = ((size_t)M + 255) / 256 * 256, lb = ((size_t)M * 4 + 255) / 256 * 256;
    uint8_t* core = reinterpret_cast<uint8_t*>(ws);
    int32_t* la = reinterpret_cast<int32_t*>(ws + mb);
    int32_t* lb_ = reinterpret_cast<int32_t*>(ws + mb + lb);
    int* flag = reinterpret_cast<int*>(ws + mb + 2 * lb);
    const unsigned grid = (unsigned)((M + CL_THREADS - 1) / CL_THREADS);
    const size_t smem = CL_THREADS * (sizeof(ClPoint) + 4 + 4 + 1);
    auto pass = [&](int mode, const int32_t* lin, int32_t* lout) {
        KBMOD_LAUNCH(cluster_pass_kernel, grid, CL_THREADS, smem, st, mode, x0y0, vxvy, nu, M, (float)ixy, (float)iv,
                     min_samples, core, lin, lout, rep, flag);
        note_launch();
    };
    pass(0, nullptr, la);
    for (int round = 0; round < M + 1; ++round) {
        if (cudaMemsetAsync(flag, 0, sizeof(int), st) != cudaSuccess) return KBMOD_ERR_CUDA;
        pass(1, la, lb_);
        KBMOD_LAUNCH(cluster_jump_kernel, grid, CL_THREADS, 0, st, core, lb_, la, M);
        note_launch();
        int changed = 0;
        if (cudaMemcpyAsync(&changed, flag, sizeof(int), cudaMemcpyDeviceToHost, st) != cudaSuccess ||
            cudaStreamSynchronize(st) != cudaSuccess)
            return KBMOD_ERR_CUDA;
        if (!changed) break;
    }
    pass(2, la, label);
    pass(3, label, nullptr);
    return cudaGetLastError() == cudaSuccess ? KBMOD_OK : KBMOD_ERR_CUDA;
}

}  // namespace kbmod
