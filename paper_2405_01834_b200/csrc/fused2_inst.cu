// fused2_inst.cu -- instantiations and launch configuration of the warp-specialised fused kernels.
#include <algorithm>

#include "fused.cuh"
#include "fused2_reg.cuh"

namespace mdb {

namespace {
F2Entry g_f2[3 * 3 * 3 * 3 * 2];
int g_f2_max_smem = 227 * 1024;
}  // namespace

F2Entry *f2_table() { return g_f2; }

// Classes with la + lb >= 2 and lc + ld >= 2 (canonical order), both outputs.
cudaError_t fused2_init(int max_smem) {
    g_f2_max_smem = max_smem;
    cudaError_t e;
#define F2_CLASS(la, lb, lc, ld) if ((e = fused2_register_##la##lb##_##lc##ld(max_smem)) != cudaSuccess) return e;
#include "fused2_classes.inc"
#undef F2_CLASS
    return cudaSuccess;
}

int fused2_dispatch(const PairView &b0, const PairView &k0, long long nq, const int32_t *qidx, int pure, int layout,
                    double *out, const double *boys_tab, int nsm, cudaStream_t st, int *info, int (*get_ws)(void *, size_t, void **), void *ws_ctx) {
    if (b0.a.l > 2 || (!b0.single && b0.b.l > 2) || k0.a.l > 2 || (!k0.single && k0.b.l > 2)) return 0;
    Fused2Args ga;
    int l[4];
    fused_make_args(b0, k0, nq, qidx, pure, layout, out, boys_tab, ga.f, l);
    const F2Entry &e = g_f2[(((l[0] * 3 + l[1]) * 3 + l[2]) * 3 + l[3]) * 2 + (pure ? 1 : 0)];
    if (!e.fn) return 0;
    // quartets per CTA: as many as shared memory and 256 consumer threads allow
    int NQ = (int)std::min<size_t>(((size_t)g_f2_max_smem - e.fixed_bytes) / e.perq_bytes, std::min<size_t>((size_t)(192 / e.nch) / e.npg, 64));
    if (NQ < 1) return 0;
    NQ = (int)std::min<long long>(NQ, std::max<long long>(1, (nq + nsm - 1) / nsm));
    ga.NQ = NQ;
    ga.TCH = (NQ * e.npg + 31) / 32 * 32;
    const int threads = e.nch * ga.TCH + MD_F2_PRODUCERS;
    const long long ngroups = (nq + NQ - 1) / NQ;
    const unsigned grid = (unsigned)std::min<long long>(ngroups, nsm);
    const size_t smem = e.perq_bytes * NQ + e.fixed_bytes;
    const int Kbra = ga.f.bra.a.K * (ga.f.bra.single ? 1 : ga.f.bra.b.K), Kket = ga.f.ket.a.K * (ga.f.ket.single ? 1 : ga.f.ket.b.K);
    const size_t need = 8 * (size_t)grid * NQ * ((size_t)Kbra * e.brec + (size_t)Kket * e.krec);
    void *ws = nullptr;
    int werr = get_ws(ws_ctx, need, &ws);
    if (werr) return werr;
    ga.scratch = (double *)ws;
    e.fn<<<grid, threads, smem, st>>>(ga);
    if (info) { info[0] = e.pb; info[1] = e.nch; info[2] = NQ; info[3] = e.nch * ga.TCH; info[4] = (int)smem; }
    return 1;
}

}  // namespace mdb
