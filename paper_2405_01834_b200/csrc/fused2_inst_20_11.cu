// fused2_inst_20_11.cu -- warp-specialised fused kernels of class (20|11), both outputs.
// One class per translation unit: with several classes in one unit the compiler stops inlining the kernel's
// local lambdas and their register arrays fall into local memory (528-byte stack frame, 1.4x slower).
#include "fused2_reg.cuh"

namespace mdb {
cudaError_t fused2_register_20_11(int max_smem) {
    cudaError_t e = f2_reg<2, 0, 1, 1, false>(max_smem);
    return e != cudaSuccess ? e : f2_reg<2, 0, 1, 1, true>(max_smem);
}
}  // namespace mdb
