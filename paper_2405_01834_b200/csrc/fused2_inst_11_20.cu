// fused2_inst_11_20.cu -- warp-specialised fused kernels of class (11|20), both outputs.
// One class per translation unit: with several classes in one unit the compiler stops inlining the kernel's
// local lambdas and their register arrays fall into local memory (528-byte stack frame, 1.4x slower).
#include "fused2_reg.cuh"

namespace mdb {
cudaError_t fused2_register_11_20(int max_smem) {
    cudaError_t e = f2_reg<1, 1, 2, 0, false>(max_smem);
    return e != cudaSuccess ? e : f2_reg<1, 1, 2, 0, true>(max_smem);
}
}  // namespace mdb
