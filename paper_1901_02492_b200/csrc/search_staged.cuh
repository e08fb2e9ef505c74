// search_staged.cuh -- interface of the shared-memory staged search kernel (search_staged.cu).
#pragma once
#include "common.cuh"

namespace kbmod {

// bytes of the device-side plan (per-block / per-image staging descriptors and offset tables)
size_t staged_plan_bytes(int N, int V, int K);

// Returns KBMOD_ERR_UNSUPPORTED when the shape does not fit the staged kernel (the caller then
// uses the direct-gather kernel).  plan_dev / enc_dev are carved from the caller's workspace.
int launch_search_staged(const float2* psiphi, const DtTable& dt, int N, int H, int W,
                         const float* vel_host, int V, int K, int min_obs, const kbmod_result& out,
                         void* plan_dev, float2* enc_dev, cudaStream_t st);

}  // namespace kbmod
