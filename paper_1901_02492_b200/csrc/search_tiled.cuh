// search_tiled.cuh -- interface of the tiled search kernels (search_tiled.cu).
#pragma once
#include <vector>

#include "common.cuh"

namespace kbmod {

// bytes of the device-side plan (per-velocity-block offset tables) for these sizes
size_t tiled_plan_bytes(int N, int V, int K);

// Host plan of the tiled kernels: per velocity block, the proven integer shift of every (velocity,
// image) pair.  Depends only on (times, velocity grid, shape, K, kernel), not on the pixel data.
struct TiledPlan {
    std::vector<int> rec;     // nblk block records (layout: search_tiled.cu)
    int nblk = 0;
    bool queued = false;      // built for search_tiledq_kernel (unproven shifts isolated in blocks of their own)
};

// Builds the plan.  KBMOD_ERR_UNSUPPORTED when the shape does not fit these kernels (the caller then
// uses the direct-gather kernel); nothing is launched or touched.
int tiled_plan_build(const DtTable& dt, int N, int H, int W, const float* vel_host, int V, int K, bool queued,
                     TiledPlan& plan);

// S3..S6 over the start rows [y_begin, y_end) with a prebuilt plan.  The result planes hold the band
// only ([(y_end - y_begin)][W][K]).  plan_dev / enc_dev are carved from the caller's workspace
// (tiled_plan_bytes() and N*H*enc_pitch(W)*8 bytes, search_common.cuh); vel_dev is the device copy of the velocity table.
// plan.queued = false: search_tiled_kernel (per-pixel lists in shared memory); true: search_tiledq_kernel
// (same gathers; survivors of the pre-test compacted into per-warp queues, lists in the output planes).
// group_w: tile columns per rasterisation group, 0 = default (kbmod_search_options.tile_group_w).
int tiled_launch(const TiledPlan& plan, const float2* psiphi, const DtTable& dt, int N, int H, int W, int K,
                 int min_obs, int y_begin, int y_end, const kbmod_result& out, void* plan_dev,
                 const float2* vel_dev, float2* enc_dev, int group_w, cudaStream_t st);

// Threshold mode (kbmod_search_threshold) on the queued kernel: the same gathers and pre-test with the
// detection threshold as the bound; survivors are scored exactly and appended to the candidate list.
// The plan must have been built with queued = true and K = 8.
int tiled_launch_threshold(const TiledPlan& plan, const float2* psiphi, const DtTable& dt, int N, int H, int W,
                           int min_obs, float nu_min, int y_begin, int y_end, const kbmod_candidates& cand,
                           unsigned long long capacity, unsigned long long* count, void* plan_dev,
                           const float2* vel_dev, float2* enc_dev, int group_w, cudaStream_t st);

// plan + launch in one call
int launch_search_tiled(const float2* psiphi, const DtTable& dt, int N, int H, int W,
                        const float* vel_host, int V, int K, int min_obs, int y_begin, int y_end,
                        const kbmod_result& out, void* plan_dev, const float2* vel_dev, float2* enc_dev,
                        bool queued, int group_w, cudaStream_t st);

}  // namespace kbmod
