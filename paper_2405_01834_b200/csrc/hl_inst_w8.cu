// hl_inst_w8.cu -- hl_kernel with 8-warp CTAs.
#include "hl_reg.cuh"
namespace mdb {
cudaError_t hl_register_w8(int max_smem, const uint32_t *herm, const double *solid) {
    cudaError_t e = upload_tables(herm, solid);
    if (e != cudaSuccess) return e;
    if ((e = hl_reg_row<1, 8>(max_smem)) != cudaSuccess) return e;
    if ((e = hl_reg_row<2, 8>(max_smem)) != cudaSuccess) return e;
    if ((e = hl_reg_row<3, 8>(max_smem)) != cudaSuccess) return e;
    return hl_reg_row<4, 8>(max_smem);
}
}  // namespace mdb
