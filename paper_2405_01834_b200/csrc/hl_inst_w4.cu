// hl_inst_w4.cu -- hl_kernel with 4-warp CTAs (small classes: several CTAs per SM).
#include "hl_reg.cuh"
namespace mdb {
cudaError_t hl_register_w4(int max_smem, const uint32_t *herm, const double *solid) {
    cudaError_t e = upload_tables(herm, solid);
    if (e != cudaSuccess) return e;
    hl_pair_table()[1] = hl_pair_kernel<1>; hl_pair_table()[2] = hl_pair_kernel<2>;
    hl_pair_table()[3] = hl_pair_kernel<3>; hl_pair_table()[4] = hl_pair_kernel<4>;
    for (int n = 1; n <= 4; ++n)
        if ((e = cudaFuncSetAttribute(hl_pair_table()[n], cudaFuncAttributeMaxDynamicSharedMemorySize, 100 * 1024)) != cudaSuccess) return e;
    if ((e = hl_reg_row<1, 4>(max_smem)) != cudaSuccess) return e;
    if ((e = hl_reg_row<2, 4>(max_smem)) != cudaSuccess) return e;
    return hl_reg_row<3, 4>(max_smem);
}
}  // namespace mdb
