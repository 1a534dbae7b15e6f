// fused_api.cuh -- what md_b200.cu sees of the fused kernels (they are compiled in fused_inst.cu).
#pragma once
#include "common.cuh"

namespace mdb {

cudaError_t fused_upload_tables(const uint32_t *herm, const double *solid);
cudaError_t fused_register_all(int max_smem);
const uint32_t *fused_rlut();   // [2*N~(24)] R-recursion LUT (device), shared with the DMMA kernels
static inline cudaError_t fused_init(int max_smem) { return fused_register_all(max_smem); }

// Returns 1 if a fused kernel was launched, 0 if the class has none, < 0 on error.
struct FusedDigest {          // exchange digestion in the kernel epilogue (fused_kernel.cuh); offsets in CALLER order a, b, c, d
    double *K; const double *D; long long n; const int32_t *off[4];
};
int fused_dispatch(const PairView &b, const PairView &k, long long nq, const int32_t *qidx, int pure, int layout,
                   double *out, const double *boys_tab, int nsm, cudaStream_t st, bool force, const FusedDigest *dg = nullptr);

// Warp-specialised fused kernels (fused2_inst.cu): same contract as fused_dispatch; info (may be null)
// receives {PB, NCH, NQ, consumer threads, smem bytes}; get_ws supplies the per-CTA pair-table scratch
// (a non-zero return value is passed back to the caller unchanged).
cudaError_t fused2_init(int max_smem);
int fused2_dispatch(const PairView &b, const PairView &k, long long nq, const int32_t *qidx, int pure, int layout,
                    double *out, const double *boys_tab, int nsm, cudaStream_t st, int *info, int (*get_ws)(void *, size_t, void **), void *ws_ctx);

}  // namespace mdb
