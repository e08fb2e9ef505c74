/*
 * kbmod_b200.h -- C ABI of the B200-native KBMOD shift-and-stack hot path.
 *
 * The calls follow the paper's statement of the problem (Whidden et al. 2019,
 * arXiv:1901.02492; citations below are PAPER.md line numbers "P:<line>"):
 *   1. kbmod_make_psi_phi : per-image likelihood images Psi_i, Phi_i   (Eq.19-20)
 *   2. kbmod_search       : exhaustive linear-trajectory search        (Eq.24-27)
 * plus the band / options / prebuilt-plan forms of the search (kbmod_search_rows,
 * kbmod_plan_create, kbmod_search_planned), a test hook (kbmod_eval_trajectories) and small
 * utilities.
 *
 * Conventions
 *   - Plain C, no torch / C++ types.  Pointers are DEVICE pointers unless marked HOST.
 *   - The library never allocates or frees caller-visible memory and never synchronises the
 *     stream (two documented exceptions: kbmod_search_status and kbmod_cluster_candidates).  The caller (PyTorch in this repo) owns every buffer and the stream.  HOST
 *     arrays are consumed before the call returns.
 *   - Images are row-major [N][H][W], x (column) fastest.  Integer coordinates are pixel
 *     centres; pixel ix covers [ix-0.5, ix+0.5).
 *   - Return value: KBMOD_OK (0) or a negative kbmod_status.  Argument errors are found
 *     before any launch; asynchronous faults surface at the caller's next synchronisation.
 *   - There is no CPU fallback: without a CUDA device every compute call returns
 *     KBMOD_ERR_CUDA.
 *   - No environment variable and no process-wide setting influences any call: what selects a
 *     kernel or tunes it is an argument (kbmod_search_options).  Calls on distinct streams with
 *     distinct workspaces are independent and thread-safe.
 *   - Deviation from the two-call signature of the problem statement, which lists vel_grid among
 *     the device arrays: vel_grid (and times) are HOST arrays here, because the library derives
 *     its per-(velocity, image) integer-shift plan from them on the host before any launch; it
 *     keeps its own device copy in the workspace.
 */
#ifndef KBMOD_B200_H
#define KBMOD_B200_H

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef enum {
    KBMOD_OK = 0,
    KBMOD_ERR_NULL = -1,        /* a required pointer is NULL */
    KBMOD_ERR_SHAPE = -2,       /* non-positive or inconsistent dimension */
    KBMOD_ERR_ARG = -3,         /* value out of range (even P, K, min_obs, non-finite time ...) */
    KBMOD_ERR_ALIGN = -4,       /* pointer not aligned as documented */
    KBMOD_ERR_CUDA = -5,        /* CUDA runtime error at launch / no device */
    KBMOD_ERR_UNSUPPORTED = -6, /* beyond the supported limits (P > 31, N > 64, K > 32) */
    KBMOD_ERR_WORKSPACE = -7,   /* workspace smaller than kbmod_search_workspace() */
    KBMOD_ERR_TIMEOUT = -8      /* a kernel gave up waiting on its own pipeline (kbmod_search_status) */
} kbmod_status;

#define KBMOD_MAX_PSF 31
#define KBMOD_MAX_IMAGES 64
#define KBMOD_MAX_K 32

/* Result planes of kbmod_search (structure of arrays).  Each member is a DEVICE pointer to
 * [H][W][K] elements, caller-owned.  For one start pixel the K slots are sorted by nu
 * descending (ties: smaller vel_idx first).  Unused slots: vel_idx = -1, n_obs = 0,
 * psi = phi = alpha = 0, nu = -INFINITY.  (Candidate record of P:241-249: start pixel =
 * plane position, velocity = vel_grid[vel_idx], likelihood nu, flux alpha.) */
typedef struct {
    int32_t* vel_idx;
    int32_t* n_obs;
    float* psi;    /* Psi_coadd, Eq.24 */
    float* phi;    /* Phi_coadd, Eq.25 */
    float* nu;     /* Psi/sqrt(Phi), Eq.26 */
    float* alpha;  /* Psi/Phi, Eq.22 */
} kbmod_result;

/*
 * Likelihood images with diagonal covariance (Eq.19-20):
 *     Psi_i(y) = sum_d  sci_i(y+d)/var_i(y+d) * T_i(d)
 *     Phi_i(y) = sum_d        1/var_i(y+d)    * T_i(d)^2       d over the P x P support
 * A pixel has zero inverse variance when it is masked, when sci or var is not finite, when
 * var <= 0, or when it lies outside the image.  If the centre pixel itself has zero
 * inverse variance (or Phi <= 0) the output is the invalid marker (psi = NaN, phi = 0).
 * This is a cross-correlation with T (Eq.19), not a convolution; they coincide for
 * point-symmetric kernels.  Arithmetic: fp32 FMAs.
 *
 *   sci, var : [N][H][W] float, device
 *   mask     : [N][H][W] uint8, device, nonzero = masked; may be NULL (no mask)
 *   psf      : HOST [N][P][P] float, psf[i][r+dy][r+dx] = T_i(dx,dy), r = (P-1)/2; taken as
 *              given (any values, not renormalised); copied before return
 *   P        : odd, 1 <= P <= KBMOD_MAX_PSF
 *   psiphi   : out, [N][H][W][2] float (psi, phi interleaved: one 8-byte sample),
 *              device, 8-byte aligned; must not alias the inputs
 *   stream   : cudaStream_t (NULL = default stream)
 */
int kbmod_make_psi_phi(const float* sci, const float* var, const uint8_t* mask,
                       const float* psf, int N, int H, int W, int P,
                       float* psiphi, void* stream);

/* Which search kernel runs (kbmod_search_options.kernel).  All return bit-identical results. */
enum {
    KBMOD_KERNEL_AUTO = 0,          /* the tiled kernel where the shape fits, else the direct-gather kernel */
    KBMOD_KERNEL_DIRECT = 1,        /* literal S3 per sample, global loads, any shape */
    KBMOD_KERNEL_TILED = 2,         /* host-proven integer shifts, global loads through L1 */
    KBMOD_KERNEL_STAGED = 3,        /* TMA-staged shared-memory windows, persistent CTAs */
    KBMOD_KERNEL_TILED_QUEUED = 4   /* the gathers of 2 with queue-compacted top-K */
};

/* Options of a search.  Zero-initialise; every field's 0 is its default; NULL = all defaults.
 * With kernel 2, 3 or 4 the call returns KBMOD_ERR_UNSUPPORTED if the shape does not fit it. */
typedef struct {
    int32_t struct_size;    /* 0 or sizeof(kbmod_search_options) */
    int32_t kernel;         /* KBMOD_KERNEL_* */
    int32_t tile_group_w;   /* kernels 2, 4: tile columns per rasterisation group, 1..256; 0 = default.
                               Changes which CTA takes which tile, never the results */
    int32_t staged_geom;    /* kernel 3: shared-memory ring geometry 0..3 (csrc/search_staged.cu) */
} kbmod_search_options;

/*
 * Exhaustive search (Eq.27).  For every start pixel (x0,y0) of image 0
 * and every velocity j of vel_grid:
 *     dt_i = (float)(times[i] - times[0])
 *     ix   = floor( fl( fl( fl(x0) + fl(vx_j*dt_i) ) + 0.5f ) )     (same for y; binary32,
 *            round-to-nearest-even, never fused; exact halves round up)
 *     an observation exists iff 0<=ix<W, 0<=iy<H and psi_i[iy][ix] is not NaN
 *     Psi = sum psi_i[iy][ix], Phi = sum phi_i[iy][ix]   fp32 adds, images in order 0..N-1
 *     eligible iff n_obs >= min_obs and Phi > 0
 *     nu = Psi/sqrt(Phi), alpha = Psi/Phi                 correctly rounded fp32
 * and the K eligible trajectories of largest nu are kept per start pixel (see kbmod_result).
 *
 *   psiphi    : [N][H][W][2] float as produced above, device, 16-byte aligned.  Contract: phi
 *               is finite and >= 0 wherever psi is not NaN; psi is finite or NaN.
 *   times     : HOST [N] double, days, finite; need not be sorted; times[0] is the start image
 *   vel_grid  : HOST [V][2] float (vx, vy) px/day, finite
 *   V >= 1; 1 <= K <= KBMOD_MAX_K; 1 <= min_obs <= N; 1 <= N <= KBMOD_MAX_IMAGES
 *   out       : HOST struct of DEVICE plane pointers, each [H][W][K], 4-byte aligned
 *   workspace : device scratch of at least kbmod_search_workspace(N,H,W,V,K) bytes,
 *               256-byte aligned; contents undefined afterwards
 */
int kbmod_search(const float* psiphi, const double* times, int N, int H, int W,
                 const float* vel_grid, int V, int K, int min_obs,
                 const kbmod_result* out, void* workspace, size_t workspace_bytes,
                 void* stream);

/*
 * kbmod_search restricted to the start rows y_begin <= y0 < y_end (0 <= y_begin <= y_end <= H), with
 * options.  Every evaluation is independent and top-K never crosses start pixels, so bands
 * of one replicated stack searched on different GPUs concatenate to the full search (row-band
 * sharding).  Trajectories still sample the whole images.
 *   out       : planes of the BAND only, each [(y_end - y_begin)][W][K]; row 0 = start row y_begin
 *               (an empty band, y_begin == y_end, writes nothing and accepts NULL planes)
 *   options   : HOST, may be NULL
 * Other arguments as kbmod_search (the workspace size does not depend on the band).
 */
int kbmod_search_rows(const float* psiphi, const double* times, int N, int H, int W,
                      const float* vel_grid, int V, int K, int min_obs, int y_begin, int y_end,
                      const kbmod_result* out, void* workspace, size_t workspace_bytes,
                      const kbmod_search_options* options, void* stream);

/*
 * The host plan of a search, built once and reused.  Everything kbmod_search derives from (times,
 * velocity grid, image shape, K, options) before it looks at a pixel -- the velocity processing
 * order, the proof that one integer shift per (velocity, image) reproduces S3 for every start pixel
 * (P:203), the staged kernel's box stream -- lives in an opaque HOST object, so repeated
 * searches of stacks taken at the same epochs with the same grid do not rebuild it.
 *   kbmod_plan_create    : argument checks as kbmod_search; *plan receives the object.  No CUDA call.
 *   kbmod_plan_kernel    : the KBMOD_KERNEL_* the plan resolved to (AUTO never remains)
 *   kbmod_search_planned : kbmod_search_rows with the plan's times / grid / shape / K / options
 *   kbmod_plan_destroy   : frees it (NULL is allowed); the plan may be destroyed as soon as the
 *                          searches using it have returned
 * A plan is immutable: any number of searches on any streams may share it concurrently.
 */
typedef struct kbmod_plan kbmod_plan;
int kbmod_plan_create(const double* times, int N, int H, int W, const float* vel_grid, int V, int K,
                      const kbmod_search_options* options, kbmod_plan** plan);
int kbmod_plan_kernel(const kbmod_plan* plan);
int kbmod_search_planned(const kbmod_plan* plan, const float* psiphi, int min_obs, int y_begin, int y_end,
                         const kbmod_result* out, void* workspace, size_t workspace_bytes, void* stream);
void kbmod_plan_destroy(kbmod_plan* plan);

/*
 * Threshold-mode search: the paper's own retention rule ("evaluate nu for all possible values
 * of y0 and v, and examine those that are above a desired detection threshold"; threshold
 * 10).  Same S3, S4, S5 and eligibility as kbmod_search; instead of the K best per start pixel,
 * EVERY eligible trajectory of the band with nu >= nu_min is appended to a compacted candidate list
 * (start pixel, velocity index, n_obs, Psi, Phi, nu, alpha).  There is no dense [H][W][K] output.
 *   out      : HOST struct of DEVICE arrays of `capacity` elements each, caller-owned
 *   count    : DEVICE counter; set to the number of trajectories found.  If it exceeds `capacity`
 *              only `capacity` of them were stored (which ones is unspecified) -- enlarge and rerun.
 *   The order of the list is unspecified; its content (as a set) is exactly the definition's.
 *   options  : kernel AUTO / DIRECT = the direct-gather kernel; TILED_QUEUED = the tiled gathers
 *              with the queue-compacted epilogue; TILED and STAGED: KBMOD_ERR_UNSUPPORTED.
 *   workspace: as kbmod_search with K = 8 (kbmod_search_workspace(N,H,W,V,8))
 */
typedef struct {
    int32_t* x;        /* start pixel */
    int32_t* y;
    int32_t* vel_idx;
    int32_t* n_obs;
    float* psi;
    float* phi;
    float* nu;
    float* alpha;
} kbmod_candidates;

int kbmod_search_threshold(const float* psiphi, const double* times, int N, int H, int W,
                           const float* vel_grid, int V, int min_obs, float nu_min, int y_begin, int y_end,
                           const kbmod_candidates* out, long long capacity, unsigned long long* count,
                           void* workspace, size_t workspace_bytes, const kbmod_search_options* options,
                           void* stream);

/*
 * Light-curve outlier filter and re-score of candidate trajectories (section 3.3: "a variation
 * on the Kalman filter ... filter out any observations that are more than five standard deviations
 * away from the best fit Kalman flux at that observation and use the remaining observations to
 * recalculate the likelihood").  The paper gives no gains or noise model; this call implements the
 * reading DESIGN.md N1-a..N1-e: light curve f_i = Psi_i/Phi_i with variance 1/Phi_i over the
 * observations that exist (S3/S4) and have Phi_i > 0; a scalar Kalman filter (state = flux,
 * random-walk process variance `process_var` per step) run forward and backward, the first
 * observation of a pass initialises it, an observation is an outlier of the pass iff
 * (f_i - x)^2 > sigma_reject^2 * (P + process_var + 1/Phi_i) and is then not ingested; the pass that
 * keeps more observations decides (tie: forward); Psi, Phi, n_obs, nu, alpha are recomputed over
 * the kept observations in image order (fp32, as kbmod_search).  All in separately rounded fp32.
 *   x0y0 : [M][2] int32 device (start pixel);  vxvy : [M][2] float device (px/day), 8-byte aligned
 *   psi, phi, nu, alpha : [M] float device;  n_obs : [M] int32 device
 *   keep : [M] uint64 device, bit i = observation i exists and was kept
 *   kalman : [M][2] float device or NULL: (flux estimate, variance) of the deciding pass
 *   nu = -INFINITY, alpha = 0 when nothing is left or Phi <= 0.
 */
int kbmod_filter_candidates(const float* psiphi, const double* times, int N, int H, int W,
                            const int32_t* x0y0, const float* vxvy, int M, float sigma_reject,
                            float process_var, float* psi, float* phi, int32_t* n_obs, float* nu,
                            float* alpha, uint64_t* keep, float* kalman, void* stream);

/*
 * Coadded postage stamps of candidate trajectories and their central moments (section 3.3:
 * "coadded postage stamps ... central moments of the images ... similarity of the moments to a
 * Gaussian centered at the middle of the stamp").  Reading DESIGN.md N2-a..N2-c:
 *   stamp[dy][dx], dy, dx in [-R, R] = mean over the observations i of the trajectory (those with
 *       bit i of keep[m] set; all when keep is NULL) of sci_i[iy_i+dy][ix_i+dx], over the images
 *       where that pixel is inside the image, unmasked and finite; 0 where none contributes.
 *   moments = (m00, cx, cy, mu20, mu02, mu11) of max(stamp, 0): total, centroid relative to the
 *       stamp centre, central second moments; all zero when m00 <= 0.
 * The accept/reject thresholds on the moments are the caller's (the paper gives none).
 *   sci : [N][H][W] float device;  mask : [N][H][W] uint8 device or NULL;  R : 0..15
 *   stamps : [M][2R+1][2R+1] float device;  moments : [M][6] float device or NULL
 */
int kbmod_coadd_stamps(const float* sci, const uint8_t* mask, const double* times, int N, int H, int W,
                       const int32_t* x0y0, const float* vxvy, const uint64_t* keep, int M, int R,
                       float* stamps, float* moments, void* stream);

/*
 * Mask builder (section 3.2; section 5.2).  A pixel of image i is detected iff sci
 * and var are finite, var > 0 and sci > sigma_thr * sqrt(var) (background 0); detections are grown
 * by the disc dx^2 + dy^2 <= grow^2 ("grown by an additional two pixels"); a pixel is static iff it
 * is grown-detected in at least min_images images ("must be masked in at least one of the other
 * science images"); mask_out_i = mask_in_i | static | (sci_i finite and > bright_counts) ("any
 * pixel in any image that exceeded 120 counts").  The paper's footprint detection is the LSST
 * stack's and is not described: this thresholding is reading DESIGN.md N3-a..N3-c.
 *   sci, var : [N][H][W] float device;  mask_in : [N][H][W] uint8 device or NULL
 *   grow : 0..8;  min_images >= 1;  mask_out : [N][H][W] uint8 device (may alias mask_in)
 */
int kbmod_build_mask(const float* sci, const float* var, const uint8_t* mask_in, int N, int H, int W,
                     float sigma_thr, int grow, int min_images, float bright_counts,
                     uint8_t* mask_out, void* stream);

/*
 * De-duplication of candidates (section 3.3: DBSCAN over the start pixel and the velocity,
 * "the highest likelihood trajectory for each group").  eps and min_samples are not given in the
 * paper; reading DESIGN.md N5-a..N5-c: candidates a, b are neighbours iff
 *     (dx^2 + dy^2)/eps_xy^2 + (dvx^2 + dvy^2)/eps_v^2 <= 1        (fp32, fixed operation order);
 * a candidate is a core point iff it has >= min_samples neighbours (itself included); clusters are
 * the connected components of the core points, labelled by their smallest core index; a non-core
 * candidate with core neighbours takes the smallest label among them, without any it is noise
 * (label -1).  rep = 1 for the member of largest nu of each cluster (ties: smaller index) and for
 * every noise candidate.
 *   x0y0 : [M][2] int32 device;  vxvy : [M][2] float device (8-byte aligned);  nu : [M] float device
 *   label : [M] int32 device;  rep : [M] uint8 device
 *   workspace : device scratch of kbmod_cluster_workspace(M) bytes, 256-byte aligned
 * All-pairs passes (O(M^2)): meant for the 1e2..1e5 candidates that survive the filters.
 * This call SYNCHRONISES the stream (label propagation runs until nothing changes).
 */
int kbmod_cluster_candidates(const int32_t* x0y0, const float* vxvy, const float* nu, int M,
                             float eps_xy, float eps_v, int min_samples, int32_t* label, uint8_t* rep,
                             void* workspace, size_t workspace_bytes, void* stream);
size_t kbmod_cluster_workspace(int M);

/* Completion status of the last kbmod_search that used this workspace.  SYNCHRONISES the stream
 * (the one call of the library that does).  KBMOD_OK, or KBMOD_ERR_TIMEOUT if a warp of the
 * TMA-staged kernel gave up a barrier wait after ~2 s (its results are then invalid; the kernel
 * terminates instead of hanging the device), or KBMOD_ERR_CUDA if the stream reports a fault. */
int kbmod_search_status(const void* workspace, void* stream);

/* Bytes of device scratch kbmod_search needs for these sizes (pure function; 0 on bad sizes). */
size_t kbmod_search_workspace(int N, int H, int W, int V, int K);

/* As kbmod_search with psi and phi given as two separate [N][H][W] float planes (the literal
 * signature of the problem statement).  They are interleaved into the workspace first, so the
 * workspace must hold kbmod_search_workspace(...) + N*H*W*8 bytes. */
int kbmod_search_split(const float* psi, const float* phi, const double* times, int N, int H,
                       int W, const float* vel_grid, int V, int K, int min_obs,
                       const kbmod_result* out, void* workspace, size_t workspace_bytes,
                       void* stream);

/*
 * The whole hot path from HOST buffers (S1..S6 plus the transfers): copies sci / var / mask to the
 * device, runs kbmod_make_psi_phi and kbmod_search, and copies the six result planes back, all
 * enqueued on `stream` (asynchronous with respect to the host when the host buffers are pinned;
 * the call itself does not synchronise).  Same arithmetic and results as the two calls above.
 *   sci, var : HOST [N][H][W] float;  mask : HOST [N][H][W] uint8 or NULL;  psf : HOST [N][P][P]
 *   times    : HOST [N] double;       vel_grid : HOST [V][2] float
 *   out      : HOST struct of HOST plane pointers, each [H][W][K]
 *   workspace: DEVICE scratch of at least kbmod_search_host_workspace(N,H,W,V,K) bytes, 256-byte
 *              aligned (holds the device copies of the inputs, psi/phi, the result planes and
 *              the search workspace); kbmod_search_status(workspace, stream) works on it too
 *   options  : HOST, may be NULL
 * Every argument error of both stages is reported before the first copy is enqueued.
 */
int kbmod_search_host(const float* sci, const float* var, const uint8_t* mask, const float* psf,
                      const double* times, int N, int H, int W, int P, const float* vel_grid, int V,
                      int K, int min_obs, const kbmod_result* out, void* workspace,
                      size_t workspace_bytes, const kbmod_search_options* options, void* stream);
size_t kbmod_search_host_workspace(int N, int H, int W, int V, int K);

/*
 * Test hook: evaluate an explicit list of M trajectories with exactly the arithmetic of
 * kbmod_search (S3 + S4), returning the coadds and every sampled pixel.
 *   x0y0 : [M][2] int32 device;  vxvy : [M][2] float device;  times : HOST [N] double
 *   Psi, Phi : [M] float device;  n_obs : [M] int32 device
 *   ixiy : [M][N][2] int32 device or NULL; (-1,-1) where the trajectory is off the image
 */
int kbmod_eval_trajectories(const float* psiphi, const double* times, int N, int H, int W,
                            const int32_t* x0y0, const float* vxvy, int M,
                            float* Psi, float* Phi, int32_t* n_obs, int32_t* ixiy,
                            void* stream);

/*
 * Test hook (host only, no CUDA call): the plan the TMA-staged kernel would execute for these
 * inputs, so that its host logic -- the proof that one integer shift per (velocity, image)
 * reproduces S3 for every start pixel, the grouping of shifted windows into shared-memory boxes,
 * the per-member offsets -- can be checked against the oracle without a GPU.
 *   times, vel_grid : HOST, as for kbmod_search;  staged_geom : as kbmod_search_options.staged_geom
 *   stream  : HOST out, nent entries of info[1] int32 each (layout: csrc/search_staged.cu)
 *   shapes  : HOST out, [nshapes][2] = (box width, box height) in samples, index = tensor-map id
 *   info    : HOST out [8] = nent, ints per entry, nshapes, tile width, tile height, velocities
 *             per block, samples per slot, header bytes
 * Returns KBMOD_ERR_WORKSPACE (with info filled) if stream_ints / max_shapes are too small.
 */
int kbmod_debug_staged_plan(const double* times, int N, int H, int W, const float* vel_grid, int V,
                            int staged_geom, int32_t* stream, size_t stream_ints, int32_t* shapes,
                            int max_shapes, int32_t* info);

/* Number of kernel launches issued by this library since load (for benchmark accounting). */
unsigned long long kbmod_launch_count(void);

/* Static description of a status code. */
const char* kbmod_status_string(int status);

/* Library version, "major.minor". */
const char* kbmod_version(void);

#ifdef __cplusplus
}
#endif
#endif /* KBMOD_B200_H */
