// hl_reg.cuh -- registry of the hl_kernel<MW, NW, warps> instantiations (one translation unit per CTA size).
#pragma once
#include "hl.cuh"

namespace mdb {

typedef void (*HlFn)(HlArgs);
typedef void (*HlPairFn)(HlPairArgs);
HlPairFn *hl_pair_table();            // [NW]
HlFn *hl_table();                     // [warps == 8][MW 0..4][NW 0..4]

template <int MW, int NW, int NWARPS>
cudaError_t hl_reg1(int max_smem) {
    auto fn = hl_kernel<MW, NW, NWARPS>;
    hl_table()[((NWARPS == 8) * 5 + MW) * 5 + NW] = fn;
    return cudaFuncSetAttribute(fn, cudaFuncAttributeMaxDynamicSharedMemorySize, max_smem);
}
template <int MW, int NWARPS>
cudaError_t hl_reg_row(int max_smem) {
    cudaError_t e;
    if ((e = hl_reg1<MW, 1, NWARPS>(max_smem)) != cudaSuccess) return e;
    if ((e = hl_reg1<MW, 2, NWARPS>(max_smem)) != cudaSuccess) return e;
    if ((e = hl_reg1<MW, 3, NWARPS>(max_smem)) != cudaSuccess) return e;
    return hl_reg1<MW, 4, NWARPS>(max_smem);
}
cudaError_t hl_register_w4(int max_smem, const uint32_t *herm, const double *solid);
cudaError_t hl_register_w8(int max_smem, const uint32_t *herm, const double *solid);

}  // namespace mdb
