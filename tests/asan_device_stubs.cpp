// Test infrastructure: the device entry points of include/fcp.h as stubs, so that the two HOST
// sources of libfcp (fcp_plan.cpp, fcp_sched.cpp) can be linked into a shared library of their
// own and run under AddressSanitizer / UndefinedBehaviorSanitizer without nvcc or a GPU
// (tests/test_sanitizers.py).  Every stub reports FCP_CUDA.
#include "fcp.h"

extern "C" {
int fcp_kv_gather(const fcp_plan*, int32_t, const void*, const void*, void*, void*, int32_t,
                  int32_t, void*, fcp_gather_counts*) { return FCP_CUDA; }
int fcp_kv_gather_piece(const fcp_plan*, int32_t, int32_t, const void*, const void*, void*, void*,
                        int32_t, int32_t, void*, fcp_gather_counts*) { return FCP_CUDA; }
int fcp_kv_scatter_add(const fcp_plan*, int32_t, const void*, const void*, int32_t, float*, float*,
                       int32_t, int32_t, void*, fcp_gather_counts*) { return FCP_CUDA; }
int fcp_kv_scatter_add_piece(const fcp_plan*, int32_t, int32_t, const void*, const void*, int32_t,
                             float*, float*, int32_t, int32_t, void*, fcp_gather_counts*) {
  return FCP_CUDA;
}
int fcp_kv_reduce_finish(const float*, const float*, void*, void*, int64_t, void*) { return FCP_CUDA; }
int fcp_sched_upload(const fcp_sched*, void*, void*) { return FCP_CUDA; }
int fcp_attn_fwd(const fcp_attn_args*) { return FCP_CUDA; }
int fcp_attn_bwd(const fcp_attn_args*, const void*, void*, void*, void*) { return FCP_CUDA; }
int fcp_attn_bwd_static(const fcp_attn_args*, const void*, void*, void*, void*) { return FCP_CUDA; }
int fcp_merge(const void*, const float*, const void*, const float*, void*, float*, int64_t, int32_t,
              int32_t, int32_t, void*) { return FCP_CUDA; }
}
