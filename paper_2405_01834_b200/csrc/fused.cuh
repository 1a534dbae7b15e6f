// fused.cuh -- registry and dispatch of the compile-time-l fused kernels (fused_kernel.cuh).
// Classes with every l <= MD_FUSED_LMAX are instantiated in canonical order (la >= lb,
// lc >= ld); other orders are served by swapping the shells of a pair and permuting the
// output strides.  3-center calls use the (la lb|lX 0) instantiation with a one-centre ket.
#pragma once
#include <vector>

#include "common.cuh"
#include "fused_kernel.cuh"

#define MD_FUSED_LMAX 2

namespace mdb {

struct FusedEntry {
    void (*fn)(FusedArgs);
    size_t smem;
    int nq;          // quartets per CTA pass
    int ctas_per_sm;
};

// [la][lb][lc][ld][pure]; only canonical entries are filled.
FusedEntry *fused_table();
void fused_make_args(const PairView &b0, const PairView &k0, long long nq, const int32_t *qidx, int pure, int layout,
                     double *out, const double *boys_tab, FusedArgs &g, int l[4]);
cudaError_t fused_register_all(int max_smem);   // defined in fused_inst.cu

template <int LA, int LB, int LC, int LD, bool PURE>
cudaError_t fused_register(int max_smem) {
    using C = FusedCfg<LA, LB, LC, LD, PURE>;
    FusedEntry &e = fused_table()[(((LA * 3 + LB) * 3 + LC) * 3 + LD) * 2 + (PURE ? 1 : 0)];
    if (C::SMEM > (size_t)max_smem) return cudaSuccess;          // stays unregistered: generic path
    auto fn = fused_kernel<LA, LB, LC, LD, PURE>;
    cudaError_t err = cudaFuncSetAttribute(fn, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)C::SMEM);
    if (err != cudaSuccess) return err;
    int nb = 0;
    err = cudaOccupancyMaxActiveBlocksPerMultiprocessor(&nb, fn, MD_FUSED_THREADS, C::SMEM);
    if (err != cudaSuccess) return err;
    e.fn = fn; e.smem = C::SMEM; e.nq = C::NQ; e.ctas_per_sm = nb > 0 ? nb : 1;
    return cudaSuccess;
}

}  // namespace mdb
