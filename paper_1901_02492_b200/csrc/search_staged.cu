// search_staged.cu -- shared-memory staged search kernel (placeholder: not built yet).
#include "search_staged.cuh"

namespace kbmod {

size_t staged_plan_bytes(int N, int V, int K) {
    (void)K;
    return (size_t)N * V * 16 + 65536;
}

int launch_search_staged(const float2*, const DtTable&, int, int, int, const float*, int, int, int,
                         const kbmod_result&, void*, float2*, cudaStream_t) {
    return KBMOD_ERR_UNSUPPORTED;
}

}  // namespace kbmod
