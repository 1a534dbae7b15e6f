// mma_api.cuh -- what md_b200.cu sees of the DMMA quartet kernels (compiled in mma_inst.cu).
#pragma once
#include "common.cuh"

namespace mdb {

struct MmaCall {
    const double *rec_bra, *rec_ket;
    long long stride_bra, stride_ket;
    int Kbra, Kket, Lb, Lk, nab, ncd;
    int kq0;
    const int32_t *qidx;
    long long nq, nket;
    double *out;
    long long s_q, s_bi, s_ki, s_ab, s_cd;
    const double *boys_tab;
    const uint32_t *rlut;
};

cudaError_t mma_init(int max_smem);
// Chooses the tile shape for the class, launches; returns cudaSuccess or the launch error.
// info (may be null) receives {MW, NW, smem bytes, cached, rslots, blk_nkb, blk_np, CTAs per SM}.
cudaError_t mma_launch(const MmaCall &c, int nsm, cudaStream_t st, int *info);

}  // namespace mdb
