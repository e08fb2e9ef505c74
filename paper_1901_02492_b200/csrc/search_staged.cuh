// search_staged.cuh -- interface of the TMA-staged search kernel (search_staged.cu).
#pragma once
#include <utility>
#include <vector>

#include "common.cuh"

namespace kbmod {

// bytes of device scratch the staged kernel needs besides the encoded stack: the entry stream
// (upper bound for these sizes)
size_t staged_plan_bytes(int N, int V);
// bytes of the encoded stack (row pitch padded to an even number of samples)
size_t staged_enc_bytes(int N, int H, int W);

// Host plan of the staged kernel: the stream of entries (one TMA box or one literal-shift step
// each) the producer warp walks per tile, and the distinct box shapes (one tensor map each).
// Depends only on (times, velocity grid, shape, ring geometry), not on the pixel data.
struct StagedPlan {
    std::vector<int> stream;                 // nent entries (layout: search_staged.cu)
    std::vector<std::pair<int, int>> shapes; // distinct (box width, box height); index = tensor-map id
    int nent = 0;
    int geom = 0;                            // ring geometry the boxes were sized for
};

// Builds the plan.  KBMOD_ERR_UNSUPPORTED when the shape does not fit this kernel; KBMOD_ERR_ARG
// for an unknown ring geometry.  Nothing is launched or touched.
int staged_plan_build(const DtTable& dt, int N, int H, int W, const float* vel_host, int V, int geom,
                      StagedPlan& plan);

// S3..S6 over the start rows [y_begin, y_end) with a prebuilt plan: host-planned integer shifts,
// TMA-staged shared-memory windows.  The result planes hold the band only.  plan_dev / enc_dev are
// carved from the caller's workspace (staged_plan_bytes() / staged_enc_bytes()); vel_dev is the
// device copy of the velocity table; status_dev is a device word the kernel sets to 1 if one of its
// barrier waits timed out.
int staged_launch(const StagedPlan& plan, const float2* psiphi, const DtTable& dt, int N, int H, int W, int K,
                  int min_obs, int y_begin, int y_end, const kbmod_result& out, void* plan_dev,
                  const float2* vel_dev, float2* enc_dev, int* status_dev, cudaStream_t st);

// plan + launch in one call
int launch_search_staged(const float2* psiphi, const DtTable& dt, int N, int H, int W,
                         const float* vel_host, int V, int K, int min_obs, int y_begin, int y_end,
                         const kbmod_result& out, void* plan_dev, const float2* vel_dev, float2* enc_dev,
                         int* status_dev, int geom, cudaStream_t st);

// Host-only: builds the entry stream for these inputs (test hook behind kbmod_debug_staged_plan).
// info[0..7] = nent, HDR_INTS, nshapes, TW, TH, B, CAP (samples per slot), HDR_BYTES.
int staged_plan_debug(const DtTable& dt, int N, int H, int W, const float* vel_host, int V, int geom,
                      int32_t* stream, size_t stream_ints, int32_t* shapes, int max_shapes, int32_t* info);

}  // namespace kbmod
