// fused.cuh -- compile-time-l fused kernels (one launch: pair setup, Boys, R, both
// contractions, solid transform, store).  Placeholder until the first fused class lands:
// every class is served by the runtime-l chain in pair.cuh + generic.cuh.
#pragma once
#include "common.cuh"

namespace mdb {

static inline cudaError_t fused_upload_tables(const uint32_t *, const double *) { return cudaSuccess; }
static inline cudaError_t fused_init(int) { return cudaSuccess; }

// Returns 1 if a fused kernel was launched, 0 if the class has none, < 0 on error.
static inline int fused_dispatch(const PairView &, const PairView &, long long, const int32_t *, int, int, double *,
                                 const double *, int, cudaStream_t, bool) {
    return 0;
}

}  // namespace mdb
