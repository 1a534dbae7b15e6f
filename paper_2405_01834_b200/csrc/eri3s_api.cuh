// eri3s_api.cuh -- what md_b200.cu sees of the one-warp-per-triplet 3-center kernel (eri3s.cuh): (ab|X) with la, lb <= 3.
#pragma once
#include "common.cuh"

namespace mdb {

cudaError_t eri3s_init(int max_smem, const uint32_t *herm, const double *solid);
bool eri3s_has_class(const PairView &b, const PairView &k);
// Returns 1 if the kernel was launched (quartet-major layout), 0 if it does not serve the class.
int eri3s_dispatch(const PairView &b, const PairView &k, long long nt, const int32_t *tidx, int pure, double *out,
                   const double *boys_tab, const uint32_t *rlut, int nsm, cudaStream_t st);

}  // namespace mdb
