// eri3s_inst.cu -- host side of the one-warp-per-triplet 3-center kernel (eri3s.cuh).
#include <algorithm>

#include "eri3s.cuh"
#include "eri3s_api.cuh"

namespace mdb {

namespace {
int g_e3_max_smem = 227 * 1024;
typedef void (*E3Fn)(Eri3sArgs);
E3Fn g_e3_fn[3][29];                          // [mode][number of ket columns]: eri3s.cuh

template <int NXC, int MODE>
cudaError_t e3_reg(int max_smem) {
    g_e3_fn[MODE][NXC] = eri3s_kernel<NXC, MODE>;
    return cudaFuncSetAttribute(eri3s_kernel<NXC, MODE>, cudaFuncAttributeMaxDynamicSharedMemorySize, max_smem);
}
// the ket pair (c, d) in the two-centre mode: what the dense per-primitive table and the register columns allow
bool e3_ket_ok(const PairView &k) {
    const int lc = k.a.l, ld = k.b.l, ncol = ncart(lc) * ncart(ld);
    if (ld == 0) return true;                                         // (c s): any l_c (sparse walk for l_c >= 5)
    return ncol <= 36 && nherm(lc + ld) * (ncol + (ncol & 1)) <= 1536;
}
bool e3_bra_ok(const PairView &b) { return b.a.l <= 3 && b.b.l <= 3; }

template <int LX>
cudaError_t e3_reg_l(int max_smem) {
    cudaError_t e = e3_reg<2 * LX + 1, 0>(max_smem);
    if (e != cudaSuccess) return e;
    if ((e = e3_reg<(LX + 1) * (LX + 2) / 2, 1>(max_smem)) != cudaSuccess) return e;
    return e3_reg<(LX + 1) * (LX + 2) / 2, 2>(max_smem);
}
}  // namespace

cudaError_t eri3s_init(int max_smem, const uint32_t *herm, const double *solid) {
    g_e3_max_smem = max_smem;
    cudaError_t e = upload_tables(herm, solid);
    if (e != cudaSuccess) return e;
    if ((e = e3_reg_l<0>(max_smem)) != cudaSuccess) return e;
    if ((e = e3_reg_l<1>(max_smem)) != cudaSuccess) return e;
    if ((e = e3_reg_l<2>(max_smem)) != cudaSuccess) return e;
    if ((e = e3_reg_l<3>(max_smem)) != cudaSuccess) return e;
    if ((e = e3_reg_l<4>(max_smem)) != cudaSuccess) return e;
    if ((e = e3_reg_l<5>(max_smem)) != cudaSuccess) return e;
    if ((e = e3_reg_l<6>(max_smem)) != cudaSuccess) return e;
    // two-centre kets (c, d) with d above s: 3 x 3, 6 x 3, 10 x 3, 6 x 6 Cartesian pairs (3, 6, 10 x 1 are registered above)
    if ((e = e3_reg<9, 2>(max_smem)) != cudaSuccess) return e;
    if ((e = e3_reg<18, 2>(max_smem)) != cudaSuccess) return e;
    if ((e = e3_reg<30, 2>(max_smem)) != cudaSuccess) return e;
    return e3_reg<36, 2>(max_smem);
}

// 3-center (ab|X) with la, lb <= 3, or a 4-center class one pair of which has l <= 3 on both shells (the kernel's bra) while the
// other (the kernel's ket) is (c s) or small enough for the dense ket table: (pp|, (dp|, (fp|, (dd| and their transposes.
bool eri3s_has_class(const PairView &b, const PairView &k) {
    if (b.single) return false;
    if (k.single) return e3_bra_ok(b);
    return (e3_bra_ok(b) && e3_ket_ok(k)) || (e3_bra_ok(k) && e3_ket_ok(b));
}

int eri3s_dispatch(const PairView &b0, const PairView &k0, long long nt, const int32_t *tidx, int pure, double *out,
                   const double *boys_tab, const uint32_t *rlut, int nsm, cudaStream_t st) {
    if (!eri3s_has_class(b0, k0)) return 0;
    const bool two = !k0.single;
    const bool swap = two && !(e3_bra_ok(b0) && e3_ket_ok(k0));                 // the caller's bra becomes the kernel's ket
    const PairView &b = swap ? k0 : b0, &k = swap ? b0 : k0;
    Eri3sArgs g;
    g.bra = b; g.X = k.a; g.D = k.b; g.kidx = two ? k.idx : nullptr; g.KD = two ? k.b.K : 1; g.lD = two ? k.b.l : 0; g.swap = swap ? 1 : 0; g.pure = pure;
    g.la = b.a.l; g.lb = b.b.l; g.lX = k.a.l; g.Ka = b.a.K; g.Kb = b.b.K; g.KX = k.a.K;
    g.nca = ncart(g.la); g.ncb = ncart(g.lb); g.nXc = two ? ncart(g.lX) * ncart(g.lD) : ncomp(g.lX, pure);
    g.nhb = nherm(g.la + g.lb); g.L = g.la + g.lb + g.lX + g.lD;
    g.tidx = tidx; g.nt = nt; g.nX = k0.npairs; g.out = out; g.boys_tab = boys_tab; g.rlut = rlut;
    const long long nab_o = (long long)ncomp(g.la, pure) * ncomp(g.lb, pure), nc_o = (long long)ncomp(g.lX, pure) * ncomp(g.lD, pure);
    g.s_t = nab_o * nc_o;
    g.s_ab = swap ? 1 : nc_o;                                  // [a][b][c][d = s]; swapped: the kernel's c is the caller's a
    g.s_c = swap ? nab_o : 1;
    auto even = [](int x) { return x + (x & 1); };
    int o = 0;
    g.o_r0 = o; o += even(nherm(g.L));
    g.o_r1 = o; o += even(g.L > 0 ? nherm(g.L - 1) : 1);
    g.o_g = o; o += even(g.nhb * g.nXc);
    g.o_acc = o; o += even(g.nca * g.ncb * g.nXc);
    g.o_e = o; o += even(3 * (g.la + 1) * (g.lb + 1) * (g.la + g.lb + 1));
    g.o_ex = o; o += even((two ? 3 : 1) * (g.lX + 1) * (g.lD + 1) * (g.lX + g.lD + 1));
    if ((two && g.nXc != 21 && g.nXc != 28) || (!two && !pure && g.nXc <= 15))
        o += nherm(g.lX + g.lD) * even(g.nXc);                                // the dense table HX[q~][col] of one ket primitive
    g.o_g0 = o; o += even(g.L + 1);
    g.per_warp = o;
    const size_t fixed = 8 * (228 + 4 * 28 * MD_HL_CSTR + 88);   // Hermite triples, four transposed solid tables, the (t,u,v) cube
    const size_t avail = (size_t)g_e3_max_smem - fixed;
    int warps = (int)std::min<size_t>(8, avail / (8 * (size_t)o));
    if (warps < 1) return 0;
    // several CTAs per SM when the slices are small: the warps of one CTA share nothing but the constant tables
    int threads = warps > 4 ? 256 : 128;
    if (warps == 8 && fixed + 8 * (size_t)o * 4 <= (size_t)g_e3_max_smem / 4) { warps = 4; threads = 128; }   // 4 CTAs of 4 warps
    g.warps = warps;
    const size_t smem = fixed + 8 * (size_t)o * warps;
    const int ctas = (int)std::max<size_t>(1, std::min<size_t>(2048 / threads, (size_t)(g_e3_max_smem + 1024) / (smem + 1024)));
    const long long nblk = (nt + warps - 1) / warps;
    const int mode = two ? 2 : pure ? 0 : 1;
    if (!g_e3_fn[mode][g.nXc]) return 0;
    g_e3_fn[mode][g.nXc]<<<(unsigned)std::min<long long>(nblk, (long long)nsm * ctas), threads, smem, st>>>(g);
    return 1;
}

}  // namespace mdb
