// fused2_inst.cu -- instantiations and launch configuration of the warp-specialised fused kernels.
#include <algorithm>

#include "fused.cuh"
#include "fused2_main.cuh"

namespace mdb {

namespace {

struct F2Entry {
    void (*fn)(Fused2Args);
    int pb, nch, npg, tb, tk, krec;
    size_t perq_bytes, fixed_bytes;   // shared memory per quartet slot and per CTA
};
F2Entry g_f2[3 * 3 * 3 * 3 * 2];
int g_f2_max_smem = 227 * 1024;

template <int LA, int LB, int LC, int LD, bool PURE, int PB, int NCH>
cudaError_t reg(int max_smem) {
    using C = F2Cfg<LA, LB, LC, LD, PURE, PB, NCH>;
    F2Entry &e = g_f2[(((LA * 3 + LB) * 3 + LC) * 3 + LD) * 2 + (PURE ? 1 : 0)];
    auto fn = fused2_kernel<LA, LB, LC, LD, PURE, PB, NCH>;
    cudaError_t err = cudaFuncSetAttribute(fn, cudaFuncAttributeMaxDynamicSharedMemorySize, max_smem);
    if (err != cudaSuccess) return err;
    e.fn = fn; e.pb = PB; e.nch = NCH; e.npg = C::NPG; e.tb = C::TB; e.tk = C::TK; e.krec = 8 + even_up(C::EPK); e.tb = 8 + even_up(C::NPB); e.fixed_bytes = C::smem_bytes(0); e.perq_bytes = C::smem_bytes(1) - e.fixed_bytes;
    return cudaSuccess;
}

}  // namespace

cudaError_t fused2_init(int max_smem) {
    g_f2_max_smem = max_smem;
    cudaError_t e;
    if ((e = reg<2, 2, 2, 2, true, 3, 2>(max_smem)) != cudaSuccess) return e;
    if ((e = reg<2, 2, 2, 2, false, 3, 2>(max_smem)) != cudaSuccess) return e;
    return cudaSuccess;
}

int fused2_dispatch(const PairView &b0, const PairView &k0, long long nq, const int32_t *qidx, int pure, int layout,
                    double *out, const double *boys_tab, int nsm, cudaStream_t st, int *info, int (*get_ws)(size_t, void **)) {
    if (b0.a.l > 2 || (!b0.single && b0.b.l > 2) || k0.a.l > 2 || (!k0.single && k0.b.l > 2)) return 0;
    Fused2Args ga;
    int l[4];
    fused_make_args(b0, k0, nq, qidx, pure, layout, out, boys_tab, ga.f, l);
    const F2Entry &e = g_f2[(((l[0] * 3 + l[1]) * 3 + l[2]) * 3 + l[3]) * 2 + (pure ? 1 : 0)];
    if (!e.fn) return 0;
    // quartets per CTA: as many as shared memory and 256 consumer threads allow
    int NQ = (int)std::min<size_t>(((size_t)g_f2_max_smem - e.fixed_bytes) / e.perq_bytes, (size_t)(192 / e.nch) / e.npg);
    if (NQ < 1) return 0;
    NQ = (int)std::min<long long>(NQ, std::max<long long>(1, (nq + nsm - 1) / nsm));
    ga.NQ = NQ;
    ga.TCH = (NQ * e.npg + 31) / 32 * 32;
    const int threads = e.nch * ga.TCH + MD_F2_PRODUCERS;
    const long long ngroups = (nq + NQ - 1) / NQ;
    const unsigned grid = (unsigned)std::min<long long>(ngroups, nsm);
    const size_t smem = e.perq_bytes * NQ + e.fixed_bytes;
    const int Kbra = ga.f.bra.a.K * (ga.f.bra.single ? 1 : ga.f.bra.b.K), Kket = ga.f.ket.a.K * (ga.f.ket.single ? 1 : ga.f.ket.b.K);
    const size_t need = 8 * (size_t)grid * NQ * ((size_t)Kbra * e.tb + (size_t)Kket * e.krec);
    void *ws = nullptr;
    int werr = get_ws(need, &ws);
    if (werr) return werr;
    ga.scratch = (double *)ws;
    e.fn<<<grid, threads, smem, st>>>(ga);
    if (info) { info[0] = e.pb; info[1] = e.nch; info[2] = NQ; info[3] = e.nch * ga.TCH; info[4] = (int)smem; }
    return 1;
}

}  // namespace mdb
