/*
 * oracle.c -- plain, slow, CPU reference of the KBMOD shift-and-stack hot path.
 *
 * TEST INFRASTRUCTURE ONLY.  Only tests/, __graft_entry__.smoke() and bench.py's
 * cpu_baseline / --impl reference legs may build, load or call this file.  The product
 * (paper_1901_02492_b200/) never links, imports or falls back to it, and it shares no
 * code, headers, tables or helpers with the CUDA path.
 *
 * Every function below is the paper's definition written as nested loops (citations are
 * PAPER.md line numbers, "P:<line>").  Readings of silent/garbled passages are the ones
 * listed in DESIGN.md section 2 ("Readings of the paper", Q1..Q19).  Pins that check this file against
 * something other than itself live in tests/test_oracle_pins.py (all pinned: P1 analytic
 * source, P2 N(0,1) noise statistics, P3 v=0 inverse-variance coadd vs numpy.average,
 * P4 independent brute force incl. the bit-level f32seq sums, P5 index-revealing images, P6 mask
 * invariants, P7 scalings).  The functions for the rows beyond the top-K search (N4 threshold
 * search, N1 light-curve filter, N3 mask builder, N2 stamps and moments; bottom of this file) are
 * pinned by tests/test_oracle_next_rows.py; where the paper gives no parameter (filter gains,
 * 5-sigma semantics, moment thresholds, footprint detection) the reading is DESIGN.md's and that
 * part is "parity unpinned" AGAINST THE PAPER -- what is pinned is that this file computes the
 * stated reading (hand-derived literals, numpy.average, scipy.ndimage, brute force).
 *
 * Build: gcc -O2 -std=c99 -ffp-contract=off -fopenmp -shared -fPIC oracle.c -lm
 *   -ffp-contract=off matters: positions and f32seq sums are defined as separately
 *   rounded binary32 operations (Q8, Q9, Q18); an FMA would change them.
 */
#include <math.h>
#include <stdint.h>
#include <stdlib.h>
#include <string.h>
#ifdef _OPENMP
#include <omp.h>
#endif

#define ORACLE_OK 0
#define ORACLE_ERR_ARG (-3)

int oracle_num_threads(void) {
#ifdef _OPENMP
    return omp_get_max_threads();
#else
    return 1;
#endif
}

void oracle_set_threads(int n) {
#ifdef _OPENMP
    if (n > 0) omp_set_num_threads(n);
#else
    (void)n;
#endif
}

/* A pixel carries information iff it is unmasked and numerically usable.
 * P:171 "we set the inverse variance to zero so that they will add nothing to the
 * likelihood sum"; non-finite or non-positive variance is read the same way (Q6). */
static int good_pixel(const float* sci, const float* var, const uint8_t* mask, size_t k) {
    if (mask && mask[k]) return 0;
    if (!isfinite(sci[k]) || !isfinite(var[k])) return 0;
    return var[k] > 0.0f;
}

/*
 * O1. Likelihood images, diagonal covariance.  P:161-167 Eq.19-20:
 *     Psi(y) = sum_x n(x) T(x - y) / sigma^2(x)
 *     Phi(y) = sum_x T(x - y)^2    / sigma^2(x)
 * written with d = x - y over the P x P support of T: a cross-correlation (Q2), terms
 * outside the image or on a not-good pixel have inverse variance 0 (Q4, Q5).
 * Sums in double, stored as binary32.  If the centre pixel itself is not good, or
 * Phi <= 0, the pixel holds the invalid marker (psi = NaN, phi = 0) (Q4).
 *
 * psf[i][r+dy][r+dx] = T_i(dx, dy).  psiphi is [N,H,W,2] (psi, phi interleaved).
 * psi_abs (optional, may be NULL): sum of |terms| of Psi, for the parity tolerance.
 */
int oracle_make_psi_phi(const float* sci, const float* var, const uint8_t* mask,
                        const float* psf, int N, int H, int W, int P,
                        float* psiphi, float* psi_abs) {
    if (!sci || !var || !psf || !psiphi) return ORACLE_ERR_ARG;
    if (N <= 0 || H <= 0 || W <= 0 || P <= 0 || (P % 2) == 0) return ORACLE_ERR_ARG;
    const int r = (P - 1) / 2;
    for (int i = 0; i < N; ++i) {
        const size_t off = (size_t)i * H * W;
        const float* s = sci + off;
        const float* v = var + off;
        const uint8_t* m = mask ? mask + off : NULL;
        const float* T = psf + (size_t)i * P * P;
#pragma omp parallel for schedule(static)
        for (int y = 0; y < H; ++y) {
            for (int x = 0; x < W; ++x) {
                double psi = 0.0, phi = 0.0, pabs = 0.0;
                for (int dy = -r; dy <= r; ++dy) {
                    const int yy = y + dy;
                    if (yy < 0 || yy >= H) continue;
                    for (int dx = -r; dx <= r; ++dx) {
                        const int xx = x + dx;
                        if (xx < 0 || xx >= W) continue;
                        const size_t k = (size_t)yy * W + xx;
                        if (!good_pixel(s, v, m, k)) continue;
                        const double t = (double)T[(dy + r) * P + (dx + r)];
                        const double term = (double)s[k] / (double)v[k] * t;
                        psi += term;
                        pabs += fabs(term);
                        phi += (1.0 / (double)v[k]) * t * t;
                    }
                }
                const size_t c = (size_t)y * W + x;
                float fpsi = (float)psi, fphi = (float)phi;
                if (!good_pixel(s, v, m, c) || !(fphi > 0.0f)) {
                    fpsi = NAN;
                    fphi = 0.0f;
                }
                psiphi[2 * (off + c)] = fpsi;
                psiphi[2 * (off + c) + 1] = fphi;
                if (psi_abs) psi_abs[off + c] = (float)pabs;
            }
        }
    }
    return ORACLE_OK;
}

/*
 * S3. Pixel hit by a linear trajectory (P:203 linear trajectories; start pixel in the
 * first image P:231; nearest pixel, Q8/Q9):
 *     f  = fl( fl(p0) + fl(v * dt) )          three separately rounded binary32 ops
 *     ip = floor( fl(f + 0.5f) )              exact halves round up
 * Returns 0 and leaves *ip alone when the pixel is outside [0, n).
 */
static int traj_pixel(int p0, float v, float dt, int n, int* ip) {
    volatile float prod = v * dt;
    volatile float f = (float)p0 + prod;
    volatile float g = f + 0.5f;
    const float fl = floorf(g);
    if (!(fl >= 0.0f && fl < (float)n)) return 0;
    *ip = (int)fl;
    return 1;
}

typedef struct {
    float Psi, Phi;
    int n_obs;
} coadd_t;

/*
 * S4. Coadded likelihood along one trajectory.  P:193-195 Eq.24-25:
 *     Psi_coadd = sum_i Psi_i(y_i),  Phi_coadd = sum_i Phi_i(y_i)
 * over the observations that exist: in bounds and not the invalid marker.
 * Images in order i = 0..N-1.  mode 0 ("f64"): sums in double, rounded once to binary32.
 * mode 1 ("f32seq"): binary32 adds in image order (Q18).
 * ixiy (optional): per-image pixel, (-1,-1) when out of bounds.
 */
static coadd_t coadd(const float* psiphi, const float* dt, int N, int H, int W,
                     int x0, int y0, float vx, float vy, int mode, int* ixiy) {
    double dPsi = 0.0, dPhi = 0.0;
    float fPsi = 0.0f, fPhi = 0.0f;
    int n = 0;
    for (int i = 0; i < N; ++i) {
        int ix = -1, iy = -1;
        const int inx = traj_pixel(x0, vx, dt[i], W, &ix);
        const int iny = traj_pixel(y0, vy, dt[i], H, &iy);
        if (ixiy) {
            ixiy[2 * i] = (inx && iny) ? ix : -1;
            ixiy[2 * i + 1] = (inx && iny) ? iy : -1;
        }
        if (!(inx && iny)) continue;
        const size_t k = 2 * (((size_t)i * H + iy) * W + ix);
        const float psi = psiphi[k], phi = psiphi[k + 1];
        if (isnan(psi)) continue;
        if (mode == 0) {
            dPsi += (double)psi;
            dPhi += (double)phi;
        } else {
            volatile float a = fPsi + psi;
            volatile float b = fPhi + phi;
            fPsi = a;
            fPhi = b;
        }
        ++n;
    }
    coadd_t c;
    c.Psi = (mode == 0) ? (float)dPsi : fPsi;
    c.Phi = (mode == 0) ? (float)dPhi : fPhi;
    c.n_obs = n;
    return c;
}

static void make_dt(const double* times, int N, float* dt) {
    /* Q7: differenced in double against image 0, rounded once to binary32 */
    for (int i = 0; i < N; ++i) dt[i] = (float)(times[i] - times[0]);
}

/* S5. P:180 Eq.22 alpha = Psi/Phi; Eq.26 nu = Psi/sqrt(Phi) (Q1).
 * binary32, correctly rounded sqrt and divisions. */
static void score(coadd_t c, float* nu, float* alpha) {
    volatile float s = sqrtf(c.Phi);
    volatile float q = c.Psi / s;
    volatile float a = c.Psi / c.Phi;
    *nu = q;
    *alpha = a;
}

typedef struct {
    float nu;
    int j;
} cand_t;

/* larger nu first; equal nu: smaller velocity index first (Q15) */
static int cand_cmp(const void* pa, const void* pb) {
    const cand_t* a = (const cand_t*)pa;
    const cand_t* b = (const cand_t*)pb;
    if (a->nu > b->nu) return -1;
    if (a->nu < b->nu) return 1;
    return (a->j > b->j) - (a->j < b->j);
}

/*
 * O2. Exhaustive search.  P:205 Eq.27 argmax over (y0, v) of nu_coadd; "evaluate
 * nu for all possible values of y0 and v"; P:231 every start pixel of the first image x
 * every grid velocity.  Retention: the K eligible trajectories of largest nu per start
 * pixel (BASELINE.json north_star; Q14), eligibility Q13, eligible <=> n_obs >= min_obs and Phi > 0.
 * Selection by a full sort of all V candidates.
 * Output planes are [(y_end - y_begin), W, K]; empty slots: vel_idx = -1, n_obs = 0,
 * psi = phi = alpha = 0, nu = -inf (Q16).
 */
int oracle_search(const float* psiphi, const double* times, int N, int H, int W,
                  const float* vel, int V, int K, int min_obs, int mode,
                  int y_begin, int y_end,
                  int32_t* o_vel, int32_t* o_nobs, float* o_psi, float* o_phi,
                  float* o_nu, float* o_alpha) {
    if (!psiphi || !times || !vel || !o_vel || !o_nobs || !o_psi || !o_phi || !o_nu || !o_alpha)
        return ORACLE_ERR_ARG;
    if (N <= 0 || H <= 0 || W <= 0 || V <= 0 || K <= 0 || min_obs < 1) return ORACLE_ERR_ARG;
    if (y_begin < 0 || y_end > H || y_begin > y_end) return ORACLE_ERR_ARG;
    float* dt = (float*)malloc(sizeof(float) * N);
    make_dt(times, N, dt);
    int err = 0;
#pragma omp parallel
    {
        cand_t* cand = (cand_t*)malloc(sizeof(cand_t) * V);
        coadd_t* acc = (coadd_t*)malloc(sizeof(coadd_t) * V);
        if (!cand || !acc) {
#pragma omp atomic write
            err = 1;
        }
#pragma omp for schedule(dynamic, 1)
        for (int y0 = y_begin; y0 < y_end; ++y0) {
            if (!cand || !acc) continue;
            for (int x0 = 0; x0 < W; ++x0) {
                int nc = 0;
                for (int j = 0; j < V; ++j) {
                    acc[j] = coadd(psiphi, dt, N, H, W, x0, y0, vel[2 * j], vel[2 * j + 1], mode, NULL);
                    if (acc[j].n_obs >= min_obs && acc[j].Phi > 0.0f) {
                        float nu, alpha;
                        score(acc[j], &nu, &alpha);
                        cand[nc].nu = nu;
                        cand[nc].j = j;
                        ++nc;
                    }
                }
                qsort(cand, nc, sizeof(cand_t), cand_cmp);
                const size_t base = ((size_t)(y0 - y_begin) * W + x0) * K;
                for (int k = 0; k < K; ++k) {
                    if (k < nc) {
                        const int j = cand[k].j;
                        float nu, alpha;
                        score(acc[j], &nu, &alpha);
                        o_vel[base + k] = j;
                        o_nobs[base + k] = acc[j].n_obs;
                        o_psi[base + k] = acc[j].Psi;
                        o_phi[base + k] = acc[j].Phi;
                        o_nu[base + k] = nu;
                        o_alpha[base + k] = alpha;
                    } else {
                        o_vel[base + k] = -1;
                        o_nobs[base + k] = 0;
                        o_psi[base + k] = 0.0f;
                        o_phi[base + k] = 0.0f;
                        o_nu[base + k] = -INFINITY;
                        o_alpha[base + k] = 0.0f;
                    }
                }
            }
        }
        free(cand);
        free(acc);
    }
    free(dt);
    return err ? ORACLE_ERR_ARG : ORACLE_OK;
}

/* O3. Dense evaluation: Psi, Phi, n_obs for every (start pixel, velocity) of a row band.
 * Planes [(y_end - y_begin), W, V].  Same loops as O2 without S5/S6. */
int oracle_eval_all(const float* psiphi, const double* times, int N, int H, int W,
                    const float* vel, int V, int mode, int y_begin, int y_end,
                    float* Psi, float* Phi, int32_t* n_obs) {
    if (!psiphi || !times || !vel || !Psi || !Phi || !n_obs) return ORACLE_ERR_ARG;
    if (N <= 0 || H <= 0 || W <= 0 || V <= 0) return ORACLE_ERR_ARG;
    if (y_begin < 0 || y_end > H || y_begin > y_end) return ORACLE_ERR_ARG;
    float* dt = (float*)malloc(sizeof(float) * N);
    make_dt(times, N, dt);
#pragma omp parallel for schedule(dynamic, 1)
    for (int y0 = y_begin; y0 < y_end; ++y0)
        for (int x0 = 0; x0 < W; ++x0)
            for (int j = 0; j < V; ++j) {
                const coadd_t c = coadd(psiphi, dt, N, H, W, x0, y0, vel[2 * j], vel[2 * j + 1], mode, NULL);
                const size_t k = ((size_t)(y0 - y_begin) * W + x0) * V + j;
                Psi[k] = c.Psi;
                Phi[k] = c.Phi;
                n_obs[k] = c.n_obs;
            }
    free(dt);
    return ORACLE_OK;
}

/* Explicit trajectory list: x0y0 [M,2] int, vxvy [M,2] float -> Psi, Phi, n_obs [M],
 * ixiy [M,N,2] (optional; (-1,-1) where the trajectory leaves the image). */
int oracle_eval_trajectories(const float* psiphi, const double* times, int N, int H, int W,
                             const int32_t* x0y0, const float* vxvy, int M, int mode,
                             float* Psi, float* Phi, int32_t* n_obs, int32_t* ixiy) {
    if (!psiphi || !times || !x0y0 || !vxvy || !Psi || !Phi || !n_obs) return ORACLE_ERR_ARG;
    if (N <= 0 || H <= 0 || W <= 0 || M < 0) return ORACLE_ERR_ARG;
    float* dt = (float*)malloc(sizeof(float) * N);
    make_dt(times, N, dt);
    for (int m = 0; m < M; ++m) {
        const coadd_t c = coadd(psiphi, dt, N, H, W, x0y0[2 * m], x0y0[2 * m + 1],
                                vxvy[2 * m], vxvy[2 * m + 1], mode,
                                ixiy ? ixiy + (size_t)m * N * 2 : NULL);
        Psi[m] = c.Psi;
        Phi[m] = c.Phi;
        n_obs[m] = c.n_obs;
    }
    free(dt);
    return ORACLE_OK;
}

/* S5 for arrays (used by the pins to score dense evaluations). */
int oracle_score(const float* Psi, const float* Phi, size_t n, float* nu, float* alpha) {
    if (!Psi || !Phi || !nu || !alpha) return ORACLE_ERR_ARG;
    for (size_t k = 0; k < n; ++k) {
        coadd_t c;
        c.Psi = Psi[k];
        c.Phi = Phi[k];
        c.n_obs = 0;
        score(c, &nu[k], &alpha[k]);
    }
    return ORACLE_OK;
}

/* =====================================================================================
 * Rows beyond the top-K search; same header rules as above.
 * ===================================================================================== */

/*
 * N4. The paper's own retention rule.  P:207 "evaluate nu for all possible values of y0 and v,
 * and examine those that are above a desired detection threshold"; P:237 threshold 10.  Every
 * eligible trajectory (n_obs >= min_obs, Phi > 0, Q13) with nu >= nu_min is emitted, in
 * (y0, x0, j) order.  Sums in f32seq mode (the decision nu >= nu_min is taken in binary32, the
 * precision of the kernels).  Returns the number found; the first `capacity` are stored.
 */
long long oracle_search_threshold(const float* psiphi, const double* times, int N, int H, int W,
                                  const float* vel, int V, int min_obs, float nu_min,
                                  int y_begin, int y_end, long long capacity,
                                  int32_t* o_x, int32_t* o_y, int32_t* o_vel, int32_t* o_nobs,
                                  float* o_psi, float* o_phi, float* o_nu, float* o_alpha) {
    if (!psiphi || !times || !vel) return ORACLE_ERR_ARG;
    if (N <= 0 || H <= 0 || W <= 0 || V <= 0 || min_obs < 1 || capacity < 0) return ORACLE_ERR_ARG;
    if (y_begin < 0 || y_end > H || y_begin > y_end) return ORACLE_ERR_ARG;
    float* dt = (float*)malloc(sizeof(float) * N);
    make_dt(times, N, dt);
    long long found = 0;
    for (int y0 = y_begin; y0 < y_end; ++y0)
        for (int x0 = 0; x0 < W; ++x0)
            for (int j = 0; j < V; ++j) {
                const coadd_t c = coadd(psiphi, dt, N, H, W, x0, y0, vel[2 * j], vel[2 * j + 1], 1, NULL);
                if (!(c.n_obs >= min_obs && c.Phi > 0.0f)) continue;
                float nu, alpha;
                score(c, &nu, &alpha);
                if (!(nu >= nu_min)) continue;
                if (found < capacity) {
                    o_x[found] = x0; o_y[found] = y0; o_vel[found] = j; o_nobs[found] = c.n_obs;
                    o_psi[found] = c.Psi; o_phi[found] = c.Phi; o_nu[found] = nu; o_alpha[found] = alpha;
                }
                ++found;
            }
    free(dt);
    return found;
}

/*
 * N1. Light-curve outlier filter and re-score.  P:241 (section 3.3): "an outlier filtering process
 * that modifies estimates of the flux and variance of an object given a sequence of observations
 * ... using the light curve of the candidate trajectory and a variation on the Kalman filter ...
 * We filter out any observations that are more than five standard deviations away from the best
 * fit Kalman flux at that observation and use the remaining observations to recalculate the
 * likelihood of the candidate."  The paper gives no gains, noise model or pass order; the reading
 * used here is DESIGN.md N1-a..N1-e (parameters: PARITY UNPINNED against the paper, the
 * arithmetic is pinned by tests/test_oracle_next_rows.py):
 *   light curve   f_i = Psi_i/Phi_i with variance r_i = 1/Phi_i (Eq.22 and the variance of
 *                 alpha) over the observations of the trajectory that exist (S3/S4) and
 *                 have Phi_i > 0, in image order;
 *   one pass      scalar Kalman filter, state = flux, random-walk process variance q per step:
 *                 first observation: x = f, P = r (kept, it cannot be tested);
 *                 then Pp = P + q, e = f - x, S = Pp + r; the observation is an outlier iff
 *                 e*e > s2*S (s2 = sigma_reject^2); an outlier is not ingested (P = Pp), otherwise
 *                 G = Pp/S, x = x + G*e, P = (1 - G)*Pp;
 *   two passes    forward (image order) and backward; the pass that keeps MORE observations
 *                 decides (tie: forward) -- a first-image outlier poisons the forward pass only;
 *   re-score      Psi, Phi, n_obs over the kept observations (observations with Phi_i <= 0 are
 *                 never tested and stay in), image order, binary32; nu, alpha by S5, or
 *                 nu = -inf, alpha = 0 when Phi <= 0 or nothing is left.
 * Every operation is one separately rounded binary32 operation in the order written (the flag is
 * a floating-point decision: both sides take it in the kernel's precision).
 * keep[m] bit i = observation i exists and was kept.  kalman[m] = (x, P) of the deciding pass.
 */
typedef struct {
    int n_kept;
    uint64_t keep;
    float x, P;
} kalman_pass_t;

static kalman_pass_t kalman_pass(const float* f, const float* r, const uint64_t usable, int N, int backward,
                                 float q, float s2) {
    kalman_pass_t o;
    o.n_kept = 0; o.keep = 0; o.x = 0.0f; o.P = 0.0f;
    int have = 0;
    volatile float x = 0.0f, P = 0.0f;
    for (int k = 0; k < N; ++k) {
        const int i = backward ? N - 1 - k : k;
        if (!((usable >> i) & 1)) continue;
        if (!have) {
            x = f[i]; P = r[i]; have = 1;
            o.keep |= (uint64_t)1 << i; ++o.n_kept;
            continue;
        }
        volatile float Pp = P + q;
        volatile float e = f[i] - x;
        volatile float S = Pp + r[i];
        volatile float ee = e * e;
        volatile float lim = s2 * S;
        if (ee > lim) {
            P = Pp;
        } else {
            volatile float G = Pp / S;
            volatile float Ge = G * e;
            volatile float xn = x + Ge;
            volatile float omg = 1.0f - G;
            volatile float Pn = omg * Pp;
            x = xn; P = Pn;
            o.keep |= (uint64_t)1 << i; ++o.n_kept;
        }
    }
    o.x = x; o.P = P;
    return o;
}

int oracle_filter_candidates(const float* psiphi, const double* times, int N, int H, int W,
                             const int32_t* x0y0, const float* vxvy, int M, float sigma_reject, float q,
                             float* o_psi, float* o_phi, int32_t* o_nobs, float* o_nu, float* o_alpha,
                             uint64_t* o_keep, float* o_kalman /* [M][2] or NULL */) {
    if (!psiphi || !times || !x0y0 || !vxvy || !o_psi || !o_phi || !o_nobs || !o_nu || !o_alpha || !o_keep)
        return ORACLE_ERR_ARG;
    if (N <= 0 || N > 64 || H <= 0 || W <= 0 || M < 0) return ORACLE_ERR_ARG;
    float* dt = (float*)malloc(sizeof(float) * N);
    make_dt(times, N, dt);
    volatile float s2v = sigma_reject * sigma_reject;
    const float s2 = s2v;
    for (int m = 0; m < M; ++m) {
        float psi[64], phi[64], f[64], r[64];
        uint64_t exists = 0, usable = 0;
        for (int i = 0; i < N; ++i) {
            int ix, iy;
            psi[i] = phi[i] = f[i] = r[i] = 0.0f;
            if (!traj_pixel(x0y0[2 * m], vxvy[2 * m], dt[i], W, &ix)) continue;
            if (!traj_pixel(x0y0[2 * m + 1], vxvy[2 * m + 1], dt[i], H, &iy)) continue;
            const size_t k = 2 * (((size_t)i * H + iy) * W + ix);
            if (isnan(psiphi[k])) continue;
            psi[i] = psiphi[k]; phi[i] = psiphi[k + 1];
            exists |= (uint64_t)1 << i;
            if (phi[i] > 0.0f) {
                volatile float fi = psi[i] / phi[i];
                volatile float ri = 1.0f / phi[i];
                f[i] = fi; r[i] = ri;
                usable |= (uint64_t)1 << i;
            }
        }
        const kalman_pass_t fw = kalman_pass(f, r, usable, N, 0, q, s2);
        const kalman_pass_t bw = kalman_pass(f, r, usable, N, 1, q, s2);
        const kalman_pass_t* best = (bw.n_kept > fw.n_kept) ? &bw : &fw;
        const uint64_t keep = (exists & ~usable) | best->keep;
        float Psi = 0.0f, Phi = 0.0f;
        int n = 0;
        for (int i = 0; i < N; ++i)
            if ((keep >> i) & 1) {
                volatile float a = Psi + psi[i];
                volatile float b = Phi + phi[i];
                Psi = a; Phi = b; ++n;
            }
        o_psi[m] = Psi; o_phi[m] = Phi; o_nobs[m] = n; o_keep[m] = keep;
        if (n > 0 && Phi > 0.0f) {
            coadd_t c; c.Psi = Psi; c.Phi = Phi; c.n_obs = n;
            score(c, &o_nu[m], &o_alpha[m]);
        } else {
            o_nu[m] = -INFINITY; o_alpha[m] = 0.0f;
        }
        if (o_kalman) { o_kalman[2 * m] = best->x; o_kalman[2 * m + 1] = best->P; }
    }
    free(dt);
    return ORACLE_OK;
}

/*
 * N3. Mask builder.  P:229 (section 3.2): sources "detected at more than 5 sigma above the
 * background" are masked, masks "grown by an additional two pixels (in radius)", and "any masked
 * pixel in a science image must be masked in at least one of the other science images" (static =
 * present at the same position in two images); "the union of the mask for all individual images"
 * is the global mask.  P:349 (section 5.2): "Any pixel in any image that exceeded 120 counts ...
 * was masked".  The footprint detection of the LSST stack is not described in the paper; reading
 * N3-a..N3-c of DESIGN.md: a pixel is detected iff sci, var finite, var > 0 and
 * sci > fl(sigma_thr * fl(sqrt(var))) (background 0: the synthetic stacks have none); grown by the
 * disc dx^2 + dy^2 <= grow^2; static iff grown-detected in >= min_images images; output
 * mask_i = mask_in_i | static | (sci_i finite and > bright_counts).  All decisions in binary32.
 */
int oracle_build_mask(const float* sci, const float* var, const uint8_t* mask_in, int N, int H, int W,
                      float sigma_thr, int grow, int min_images, float bright_counts, uint8_t* mask_out) {
    if (!sci || !var || !mask_out) return ORACLE_ERR_ARG;
    if (N <= 0 || H <= 0 || W <= 0 || grow < 0 || min_images < 1) return ORACLE_ERR_ARG;
    const size_t npx = (size_t)H * W;
    uint8_t* det = (uint8_t*)calloc(npx, 1);
    int* cnt = (int*)calloc(npx, sizeof(int));
    for (int i = 0; i < N; ++i) {
        const float* s = sci + i * npx;
        const float* v = var + i * npx;
        for (size_t k = 0; k < npx; ++k) {
            det[k] = 0;
            if (isfinite(s[k]) && isfinite(v[k]) && v[k] > 0.0f) {
                volatile float sd = sqrtf(v[k]);
                volatile float lim = sigma_thr * sd;
                det[k] = s[k] > lim;
            }
        }
        for (int y = 0; y < H; ++y)
            for (int x = 0; x < W; ++x) {
                int g = 0;
                for (int dy = -grow; dy <= grow && !g; ++dy)
                    for (int dx = -grow; dx <= grow && !g; ++dx) {
                        if (dx * dx + dy * dy > grow * grow) continue;
                        const int yy = y + dy, xx = x + dx;
                        if (yy < 0 || yy >= H || xx < 0 || xx >= W) continue;
                        g = det[(size_t)yy * W + xx];
                    }
                cnt[(size_t)y * W + x] += g;
            }
    }
    for (int i = 0; i < N; ++i)
        for (size_t k = 0; k < npx; ++k) {
            const float s = sci[i * npx + k];
            int m = mask_in ? (mask_in[i * npx + k] != 0) : 0;
            m |= cnt[k] >= min_images;
            m |= isfinite(s) && s > bright_counts;
            mask_out[i * npx + k] = (uint8_t)m;
        }
    free(det);
    free(cnt);
    return ORACLE_OK;
}

/*
 * N2. Coadded postage stamps and their central moments.  P:243 (section 3.3): "we build coadded
 * postage stamps for all remaining candidate trajectories ... calculate the central moments of
 * the images and filter based upon the similarity of the moments to a Gaussian centered at the
 * middle of the stamp."  Reading N2-a..N2-c of DESIGN.md (thresholds: PARITY UNPINNED against the
 * paper, which gives none):
 *   stamp   for dy, dx in [-R, R]: mean over the kept observations i (bit i of keep) of
 *           sci_i[iy_i + dy][ix_i + dx], taken over the images where that pixel is inside the
 *           image, unmasked and finite; 0 where no image contributes.  Sum in image order in
 *           binary32, one division by the count.
 *   moments on w = max(stamp, 0), row-major binary32 accumulation, each product and sum
 *           separately rounded: m00 = sum w; cx = (sum w*dx)/m00, cy = (sum w*dy)/m00;
 *           mu20 = (sum w*(dx-cx)^2)/m00, mu02, mu11 likewise.  m00 <= 0 -> all zero.
 * stamps [M][2R+1][2R+1]; moments [M][6] = (m00, cx, cy, mu20, mu02, mu11).
 */
int oracle_coadd_stamps(const float* sci, const uint8_t* mask, const double* times, int N, int H, int W,
                        const int32_t* x0y0, const float* vxvy, const uint64_t* keep, int M, int R,
                        float* stamps, float* moments) {
    if (!sci || !times || !x0y0 || !vxvy || !stamps) return ORACLE_ERR_ARG;
    if (N <= 0 || N > 64 || H <= 0 || W <= 0 || M < 0 || R < 0) return ORACLE_ERR_ARG;
    const int S = 2 * R + 1;
    float* dt = (float*)malloc(sizeof(float) * N);
    make_dt(times, N, dt);
    for (int m = 0; m < M; ++m) {
        int ix[64], iy[64], on[64];
        for (int i = 0; i < N; ++i) {
            on[i] = traj_pixel(x0y0[2 * m], vxvy[2 * m], dt[i], W, &ix[i]) &&
                    traj_pixel(x0y0[2 * m + 1], vxvy[2 * m + 1], dt[i], H, &iy[i]) &&
                    (!keep || ((keep[m] >> i) & 1));
        }
        float* st = stamps + (size_t)m * S * S;
        for (int dy = -R; dy <= R; ++dy)
            for (int dx = -R; dx <= R; ++dx) {
                float sum = 0.0f;
                int n = 0;
                for (int i = 0; i < N; ++i) {
                    if (!on[i]) continue;
                    const int yy = iy[i] + dy, xx = ix[i] + dx;
                    if (yy < 0 || yy >= H || xx < 0 || xx >= W) continue;
                    const size_t k = ((size_t)i * H + yy) * W + xx;
                    if ((mask && mask[k]) || !isfinite(sci[k])) continue;
                    volatile float a = sum + sci[k];
                    sum = a; ++n;
                }
                volatile float mean = n ? sum / (float)n : 0.0f;
                st[(dy + R) * S + (dx + R)] = mean;
            }
        if (!moments) continue;
        float* mo = moments + (size_t)m * 6;
        volatile float m00 = 0.0f, sx = 0.0f, sy = 0.0f;
        for (int dy = -R; dy <= R; ++dy)
            for (int dx = -R; dx <= R; ++dx) {
                const float w = fmaxf(st[(dy + R) * S + (dx + R)], 0.0f);
                volatile float wx = w * (float)dx, wy = w * (float)dy;
                m00 = m00 + w; sx = sx + wx; sy = sy + wy;
            }
        if (!(m00 > 0.0f)) { for (int k = 0; k < 6; ++k) mo[k] = 0.0f; continue; }
        volatile float cx = sx / m00, cy = sy / m00;
        volatile float s20 = 0.0f, s02 = 0.0f, s11 = 0.0f;
        for (int dy = -R; dy <= R; ++dy)
            for (int dx = -R; dx <= R; ++dx) {
                const float w = fmaxf(st[(dy + R) * S + (dx + R)], 0.0f);
                volatile float ux = (float)dx - cx, uy = (float)dy - cy;
                volatile float wux = w * ux, wuy = w * uy;
                volatile float a = wux * ux, b = wuy * uy, c = wux * uy;
                s20 = s20 + a; s02 = s02 + b; s11 = s11 + c;
            }
        volatile float mu20 = s20 / m00, mu02 = s02 / m00, mu11 = s11 / m00;
        mo[0] = m00; mo[1] = cx; mo[2] = cy; mo[3] = mu20; mo[4] = mu02; mo[5] = mu11;
    }
    free(dt);
    return ORACLE_OK;
}

/*
 * N5. De-duplication of candidates by DBSCAN.  P:249 (section 3.3): "We take the starting x and y
 * pixels and the horizontal and vertical velocities of the candidate trajectories and use the DBSCAN
 * clustering method (Ester et al. 1996) ... to group similar trajectories.  We then take the highest
 * likelihood trajectory for each group".  eps and min_samples are not given (PARITY UNPINNED against
 * the paper); reading N5-a..N5-c of DESIGN.md:
 *   neighbours   a, b are neighbours iff d2 <= 1 with
 *                d2 = fl( fl(fl(dx*dx + dy*dy) * ixy) + fl(fl(fl(dvx*dvx) + fl(dvy*dvy)) * iv) ),
 *                dx, dy exact integers, dvx = fl(vx_a - vx_b), ixy = fl(1/fl(eps_xy^2)), iv = fl(1/fl(eps_v^2));
 *                every point is its own neighbour;
 *   DBSCAN       core iff it has >= min_samples neighbours; clusters = connected components of the core
 *                points; label = smallest index of a core point of the component (canonical, unique);
 *                a non-core point with core neighbours takes the smallest label among them (DBSCAN
 *                leaves this choice open); without any it is noise, label -1;
 *   keep         rep = 1 for the member of each cluster with the largest nu (ties: smaller index) and
 *                for every noise point.
 */
static int cl_neighbours(const int32_t* xy, const float* v, int a, int b, float ixy, float iv) {
    const long long dx = (long long)xy[2 * a] - xy[2 * b], dy = (long long)xy[2 * a + 1] - xy[2 * b + 1];
    volatile float r2 = (float)(dx * dx + dy * dy);
    volatile float dvx = v[2 * a] - v[2 * b], dvy = v[2 * a + 1] - v[2 * b + 1];
    volatile float sx = dvx * dvx, sy = dvy * dvy;
    volatile float v2 = sx + sy;
    volatile float ta = r2 * ixy, tb = v2 * iv;
    volatile float d2 = ta + tb;
    return d2 <= 1.0f;
}

int oracle_cluster_candidates(const int32_t* x0y0, const float* vxvy, const float* nu, int M, float eps_xy,
                              float eps_v, int min_samples, int32_t* label, uint8_t* rep) {
    if (M < 0 || (M > 0 && (!x0y0 || !vxvy || !nu || !label || !rep))) return ORACLE_ERR_ARG;
    if (!(eps_xy > 0.0f) || !(eps_v > 0.0f) || min_samples < 1) return ORACLE_ERR_ARG;
    volatile float exy2 = eps_xy * eps_xy, ev2 = eps_v * eps_v;
    volatile float ixy = 1.0f / exy2, iv = 1.0f / ev2;
    uint8_t* core = (uint8_t*)calloc(M ? M : 1, 1);
    for (int i = 0; i < M; ++i) {
        int n = 0;
        for (int j = 0; j < M; ++j) n += cl_neighbours(x0y0, vxvy, i, j, ixy, iv);
        core[i] = n >= min_samples;
        label[i] = -1;
    }
    int* stack = (int*)malloc(sizeof(int) * (M ? M : 1));
    for (int s = 0; s < M; ++s) {                       /* components in order of their smallest core index */
        if (!core[s] || label[s] >= 0) continue;
        int top = 0;
        stack[top++] = s;
        label[s] = s;
        while (top) {
            const int i = stack[--top];
            for (int j = 0; j < M; ++j)
                if (core[j] && label[j] < 0 && cl_neighbours(x0y0, vxvy, i, j, ixy, iv)) {
                    label[j] = s;
                    stack[top++] = j;
                }
        }
    }
    for (int i = 0; i < M; ++i) {
        if (core[i]) continue;
        int best = -1;
        for (int j = 0; j < M; ++j)
            if (core[j] && cl_neighbours(x0y0, vxvy, i, j, ixy, iv) && (best < 0 || label[j] < best)) best = label[j];
        label[i] = best;
    }
    for (int i = 0; i < M; ++i) {
        int r = 1;
        if (label[i] >= 0)
            for (int j = 0; j < M && r; ++j)
                if (j != i && label[j] == label[i] && (nu[j] > nu[i] || (nu[j] == nu[i] && j < i))) r = 0;
        rep[i] = (uint8_t)r;
    }
    free(stack);
    free(core);
    return ORACLE_OK;
}
