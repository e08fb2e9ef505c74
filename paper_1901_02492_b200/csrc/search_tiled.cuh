// search_tiled.cuh -- interface of the tiled search kernel (search_tiled.cu).
#pragma once
#include "common.cuh"

namespace kbmod {

// bytes of the device-side plan (per-velocity-block offset tables) for these sizes
size_t tiled_plan_bytes(int N, int V, int K);

// S3..S6 with host-planned integer shifts.  Returns KBMOD_ERR_UNSUPPORTED when the shape does not
// fit this kernel (the caller then uses the direct-gather kernel).  plan_dev / enc_dev are carved
// from the caller's workspace (tiled_plan_bytes() and N*H*W*8 bytes); vel_dev is the device copy of the velocity table.
// queued = false: search_tiled_kernel (per-pixel lists in shared memory); true: search_tiledq_kernel
// (same gathers; survivors of the pre-test compacted into per-warp queues, lists in the output planes).
int launch_search_tiled(const float2* psiphi, const DtTable& dt, int N, int H, int W,
                        const float* vel_host, int V, int K, int min_obs, const kbmod_result& out,
                        void* plan_dev, const float2* vel_dev, float2* enc_dev, bool queued, cudaStream_t st);

}  // namespace kbmod
