// placeholder replaced below
#include "common.cuh"
namespace sharq {
struct LinearArgs;
sharq_status launch_linear(const sharq_config*, const LinearArgs&, int32_t, const int32_t*, void*, size_t, int, cudaStream_t) { return SHARQ_EINVAL; }
size_t linear_workspace_bytes(const sharq_config*, int64_t, int64_t, int64_t, int32_t) { return 0; }
}
