// lowl_api.cuh -- what md_b200.cu sees of the one-thread-per-quartet kernel for the classes with every l <= 1.
#pragma once
#include "common.cuh"

namespace mdb {

cudaError_t lowl_init(int max_smem);
bool lowl_has_class(const PairView &b, const PairView &k);
// Returns 1 if the kernel was launched (quartet-major layout), 0 if the class has none.
int lowl_dispatch(const PairView &b, const PairView &k, long long nq, const int32_t *qidx, int pure, double *out,
                  const double *boys_tab, int nsm, cudaStream_t st);

}  // namespace mdb
