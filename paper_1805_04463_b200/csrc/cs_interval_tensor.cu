// cs_interval_tensor.cu -- stage a2, tensor route (placeholder until the tcgen05 kernel lands).
#include "cs_common.cuh"

namespace cs {

bool interval_tensor_available() { return false; }
size_t interval_tensor_scratch_bytes(int64_t, int64_t) { return 0; }
int launch_interval_tensor(const uint64_t *, const uint64_t *, int64_t, int64_t, int64_t, int64_t, int64_t,
                           int64_t *, int64_t *, void *, size_t, cudaStream_t)
{
    return CS_ERR_ARG;
}

}  // namespace cs
