// fused2_inst_22_22.cu -- warp-specialised fused kernels of class (22|22), both outputs.
// One class per translation unit: with several classes in one unit the compiler stops inlining the kernel's
// local lambdas and their register arrays fall into local memory (528-byte stack frame, 1.4x slower).
#include "fused2_reg.cuh"

namespace mdb {
cudaError_t fused2_register_22_22(int max_smem) {
    cudaError_t e = f2_reg<2, 2, 2, 2, false>(max_smem);
    return e != cudaSuccess ? e : f2_reg<2, 2, 2, 2, true>(max_smem);
}
}  // namespace mdb
