// hl_api.cuh -- what md_b200.cu sees of the high-l quartet kernel (compiled in hl_inst*.cu).
#pragma once
#include "common.cuh"

namespace mdb {

struct HlCall {
    PairView bra, ket;
    int pure;
    const int32_t *qidx;
    long long nq;
    double *out;
    long long s_q, s_bi, s_ki, s_ab, s_cd;
    const double *boys_tab;
    const uint32_t *rlut;
};

cudaError_t hl_init(int max_smem, const uint32_t *herm, const double *solid);
// Tile shape, shared-memory carve-up and grid for this call.  Returns 0 if the kernel does not serve the (class, K)
// (it then falls to the runtime-l chain), else 1 and the scratch the launch needs in *scratch_bytes.
int hl_plan(const HlCall &c, int nsm, size_t *scratch_bytes);
// Launch with the plan of the same call; scratch = device buffer of *scratch_bytes.  info (may be null) receives
// {MW, NW, warps, smem bytes, CTAs per SM, row passes, S1 mode (0 in-kernel, 1 per pair, 2 per quartet chunk), grid};
// launches = kernels enqueued.
cudaError_t hl_launch(const HlCall &c, int nsm, void *scratch, cudaStream_t st, int *info, int *launches);

}  // namespace mdb
