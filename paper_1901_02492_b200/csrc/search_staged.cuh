// search_staged.cuh -- interface of the TMA-staged search kernel (search_staged.cu).
#pragma once
#include "common.cuh"

namespace kbmod {

// bytes of device scratch the staged kernel needs besides the encoded stack: the entry stream
// (upper bound for these sizes)
size_t staged_plan_bytes(int N, int V);
// bytes of the encoded stack (row pitch padded to an even number of samples)
size_t staged_enc_bytes(int N, int H, int W);

// S3..S6 with host-planned integer shifts and TMA-staged shared-memory windows.  Returns
// KBMOD_ERR_UNSUPPORTED when the shape does not fit this kernel (the caller then uses the
// direct-gather kernel).  plan_dev / enc_dev are carved from the caller's workspace
// (staged_plan_bytes() / staged_enc_bytes()); vel_dev is the device copy of the velocity table;
// status_dev is a device word the kernel sets to 1 if one of its barrier waits timed out.
int launch_search_staged(const float2* psiphi, const DtTable& dt, int N, int H, int W,
                         const float* vel_host, int V, int K, int min_obs, const kbmod_result& out,
                         void* plan_dev, const float2* vel_dev, float2* enc_dev, int* status_dev, cudaStream_t st);

// Host-only: builds the entry stream for these inputs (test hook behind kbmod_debug_staged_plan).
// info[0..7] = nent, HDR_INTS, nshapes, TW, TH, B, CAP (samples per slot), HDR_BYTES.
int staged_plan_debug(const DtTable& dt, int N, int H, int W, const float* vel_host, int V,
                      int32_t* stream, size_t stream_ints, int32_t* shapes, int max_shapes, int32_t* info);

}  // namespace kbmod
