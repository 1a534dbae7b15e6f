// fused2_reg.cuh -- registry of the warp-specialised fused kernels; one translation unit per bra pair
// instantiates its classes (generated from fused2_classes.inc by build.py), fused2_inst.cu holds the table and the launch logic.
#pragma once
#include "fused2_main.cuh"

namespace mdb {

struct F2Entry {
    void (*fn)(Fused2Args);
    int pb, nch, npg, brec, krec;     // tile shape; scratch record sizes (doubles) of a bra / ket primitive pair
    size_t perq_bytes, fixed_bytes;   // shared memory per quartet slot and per CTA
};
F2Entry *f2_table();                  // [la][lb][lc][ld][pure], canonical order only

// Tile shape by class: two cd chunks when the first ket shell has 6 Cartesians, and as many Hermite rows per
// thread as keep the accumulators within 54 registers pairs.
template <int LC, int LD>
constexpr int f2_nch() { return ncart(LC) >= 6 ? 2 : 1; }
template <int LC, int LD>
constexpr int f2_pb() {
    constexpr int nacc = (ncart(LC) + f2_nch<LC, LD>() - 1) / f2_nch<LC, LD>() * ncart(LD);
    return 3 * nacc <= 54 ? 3 : 2 * nacc <= 54 ? 2 : 1;
}

template <int LA, int LB, int LC, int LD, bool PURE>
cudaError_t f2_reg(int max_smem) {
    constexpr int PB = f2_pb<LC, LD>(), NCH = f2_nch<LC, LD>();
    using C = F2Cfg<LA, LB, LC, LD, PURE, PB, NCH>;
    F2Entry &e = f2_table()[(((LA * 3 + LB) * 3 + LC) * 3 + LD) * 2 + (PURE ? 1 : 0)];
    auto fn = fused2_kernel<LA, LB, LC, LD, PURE, PB, NCH>;
    cudaError_t err = cudaFuncSetAttribute(fn, cudaFuncAttributeMaxDynamicSharedMemorySize, max_smem);
    if (err != cudaSuccess) return err;
    e.fn = fn; e.pb = PB; e.nch = NCH; e.npg = C::NPG;
    e.brec = 8 + even_up(C::NPB); e.krec = 8 + even_up(C::EPK);
    e.fixed_bytes = C::smem_bytes(0); e.perq_bytes = C::smem_bytes(1) - e.fixed_bytes;
    return cudaSuccess;
}

// one registration function per class, each in its own generated translation unit (fused2_classes.inc, build.py)
#define F2_CLASS(la, lb, lc, ld) cudaError_t fused2_register_##la##lb##_##lc##ld(int max_smem);
#include "fused2_classes.inc"
#undef F2_CLASS

}  // namespace mdb
