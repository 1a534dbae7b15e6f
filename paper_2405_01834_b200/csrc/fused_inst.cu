// fused_inst.cu -- instantiations of the fused kernels (canonical classes, l <= MD_FUSED_LMAX).
#include "fused.cuh"
#include "fused_api.cuh"

namespace mdb {

static FusedEntry g_table[3 * 3 * 3 * 3 * 2];
FusedEntry *fused_table() { return g_table; }

static uint32_t *g_rlut = nullptr;
const uint32_t *fused_rlut() { return g_rlut; }

cudaError_t fused_upload_tables(const uint32_t *herm, const double *solid) {
    cudaError_t e = upload_tables(herm, solid);
    if (e != cudaSuccess) return e;
    // R-recursion LUT (Eq. 24): for Hermite entry e = (t,u,v) of the degree-sorted list,
    // word 0 = i1 | i2 << 12 | axis << 24 | coef << 26 with
    //   [e]^(m) = PQ[axis] * [i1]^(m+1) + coef * [i2]^(m+1),  i1 = e - 1_axis, i2 = e - 2_axis, coef = e_axis - 1
    // on the first axis with a non-zero index; word 1 = packed (t,u,v,n).
    std::vector<uint32_t> lut(2 * MD_NHERM_MAX);
    for (int k = 0; k < MD_NHERM_MAX; ++k) {
        int t = herm[k] & 0xff, u = herm[k] >> 8 & 0xff, v = herm[k] >> 16 & 0xff;
        uint32_t w = 0;
        if (t > 0) w = herm_index(t - 1, u, v) | (t > 1 ? herm_index(t - 2, u, v) : 0) << 12 | 0u << 24 | (uint32_t)(t - 1) << 26;
        else if (u > 0) w = herm_index(t, u - 1, v) | (u > 1 ? herm_index(t, u - 2, v) : 0) << 12 | 1u << 24 | (uint32_t)(u - 1) << 26;
        else if (v > 0) w = herm_index(t, u, v - 1) | (v > 1 ? herm_index(t, u, v - 2) : 0) << 12 | 2u << 24 | (uint32_t)(v - 1) << 26;
        lut[2 * k] = w;
        lut[2 * k + 1] = herm[k];               // t | u<<8 | v<<16 | n<<24
    }
    if (!g_rlut) {
        e = cudaMalloc(&g_rlut, lut.size() * sizeof(uint32_t));
        if (e != cudaSuccess) return e;
    }
    return cudaMemcpy(g_rlut, lut.data(), lut.size() * sizeof(uint32_t), cudaMemcpyHostToDevice);
}

#define REG(a, b, c, d)                                                     \
    if ((e = fused_register<a, b, c, d, false>(max_smem)) != cudaSuccess) return e; \
    if ((e = fused_register<a, b, c, d, true>(max_smem)) != cudaSuccess) return e;
#define REG_KET(a, b) REG(a, b, 0, 0) REG(a, b, 1, 0) REG(a, b, 1, 1) REG(a, b, 2, 0) REG(a, b, 2, 1) REG(a, b, 2, 2)

cudaError_t fused_register_all(int max_smem) {
    cudaError_t e;
    REG_KET(0, 0) REG_KET(1, 0) REG_KET(1, 1) REG_KET(2, 0) REG_KET(2, 1) REG_KET(2, 2)
    return cudaSuccess;
}

}  // namespace mdb

namespace mdb {

// Canonical order (la >= lb, lc >= ld) and output strides for a fused launch; l[] receives the kernel's class.
void fused_make_args(const PairView &b0, const PairView &k0, long long nq, const int32_t *qidx, int pure, int layout,
                     double *out, const double *boys_tab, FusedArgs &g, int l[4]) {
    PairView b = b0, k = k0;
    int la = b.a.l, lb = b.single ? 0 : b.b.l, lc = k.a.l, ld = k.single ? 0 : k.b.l;
    // caller's component strides (include/md_b200.h layouts)
    const long long na = ncomp(la, pure), nb = ncomp(lb, pure), nc = ncomp(lc, pure), nd = ncomp(ld, pure);
    const long long nab = na * nb, ncd = nc * nd;
    long long ca, cb, cc, cd;
    if (layout == 1) {                               // MD_LAYOUT_PAPER: ij + nbra*(ab + N_ab*(cd + N_cd*kl))
        const long long nbra = b.npairs;
        ca = nbra * nb; cb = nbra; cc = nbra * nab * nd; cd = nbra * nab;
        g.s_q = 0; g.s_bi = 1; g.s_ki = nbra * nab * ncd;
    } else {
        ca = nb * ncd; cb = ncd; cc = nd; cd = 1;
        if (qidx) { g.s_q = nab * ncd; g.s_bi = 0; g.s_ki = 0; }
        else { g.s_q = 0; g.s_bi = k.npairs * nab * ncd; g.s_ki = nab * ncd; }
    }
    g.bra_swap = 0; g.ket_swap = 0;
    if (!b.single && la < lb) { std::swap(b.a, b.b); std::swap(la, lb); std::swap(ca, cb); g.bra_swap = 1; }
    if (!k.single && lc < ld) { std::swap(k.a, k.b); std::swap(lc, ld); std::swap(cc, cd); g.ket_swap = 1; }
    g.bra = b; g.ket = k; g.qidx = qidx; g.nq = nq; g.nket = k.npairs; g.out = out;
    g.sa = ca; g.sb = cb; g.sc = cc; g.sd = cd;
    g.boys_tab = boys_tab; g.rlut = g_rlut;
    l[0] = la; l[1] = lb; l[2] = lc; l[3] = ld;
}

int fused_dispatch(const PairView &b0, const PairView &k0, long long nq, const int32_t *qidx, int pure, int layout,
                   double *out, const double *boys_tab, int nsm, cudaStream_t st, bool /*force*/, const FusedDigest *dg) {
    if (b0.a.l > MD_FUSED_LMAX || (!b0.single && b0.b.l > MD_FUSED_LMAX) || k0.a.l > MD_FUSED_LMAX ||
        (!k0.single && k0.b.l > MD_FUSED_LMAX))
        return 0;
    FusedArgs g;
    int l[4];
    fused_make_args(b0, k0, nq, qidx, pure, layout, out, boys_tab, g, l);
    const FusedEntry &e = g_table[(((l[0] * 3 + l[1]) * 3 + l[2]) * 3 + l[3]) * 2 + (pure ? 1 : 0)];
    if (!e.fn) return 0;
    if (dg) {                                            // kernel order: (b,a) / (d,c) when the pair was swapped
        g.dg_K = dg->K; g.dg_D = dg->D; g.dg_n = dg->n;
        g.dg_off[0] = dg->off[g.bra_swap ? 1 : 0]; g.dg_off[1] = dg->off[g.bra_swap ? 0 : 1];
        g.dg_off[2] = dg->off[g.ket_swap ? 3 : 2]; g.dg_off[3] = dg->off[g.ket_swap ? 2 : 3];
    }
    const long long ngroups = (nq + e.nq - 1) / e.nq;
    const unsigned grid = (unsigned)std::min<long long>(ngroups, (long long)nsm * e.ctas_per_sm);
    e.fn<<<grid, MD_FUSED_THREADS, e.smem, st>>>(g);
    return 1;
}

}  // namespace mdb
