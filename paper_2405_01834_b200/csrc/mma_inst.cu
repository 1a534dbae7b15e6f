// mma_inst.cu -- instantiations of eri_mma_kernel<MW, NW> and the host-side tile selection.
#include <algorithm>

#include "mma.cuh"
#include "mma_api.cuh"

namespace mdb {

namespace {

constexpr int MWMAX = 5, NWMAX = 4;
typedef void (*MmaFn)(MmaArgs);
MmaFn g_fn[2][MWMAX + 1][NWMAX + 1];      // [0]: 4-warp CTAs, [1]: 8-warp CTAs
int g_max_smem = 227 * 1024;

template <int MW, int NW>
cudaError_t reg1(int max_smem) {
    g_fn[0][MW][NW] = eri_mma_kernel<MW, NW, 4>;
    g_fn[1][MW][NW] = eri_mma_kernel<MW, NW, 8>;
    cudaError_t e = cudaFuncSetAttribute(eri_mma_kernel<MW, NW, 4>, cudaFuncAttributeMaxDynamicSharedMemorySize, max_smem - 1024);
    if (e != cudaSuccess) return e;
    return cudaFuncSetAttribute(eri_mma_kernel<MW, NW, 8>, cudaFuncAttributeMaxDynamicSharedMemorySize, max_smem - 1024);
}
template <int MW>
cudaError_t reg_row(int max_smem) {
    cudaError_t e;
    if ((e = reg1<MW, 1>(max_smem)) != cudaSuccess) return e;
    if ((e = reg1<MW, 2>(max_smem)) != cudaSuccess) return e;
    if ((e = reg1<MW, 3>(max_smem)) != cudaSuccess) return e;
    return reg1<MW, 4>(max_smem);
}

}  // namespace

cudaError_t mma_init(int max_smem) {
    g_max_smem = max_smem;
    cudaError_t e;
    if ((e = reg_row<1>(max_smem)) != cudaSuccess) return e;
    if ((e = reg_row<2>(max_smem)) != cudaSuccess) return e;
    if ((e = reg_row<3>(max_smem)) != cudaSuccess) return e;
    if ((e = reg_row<4>(max_smem)) != cudaSuccess) return e;
    return reg_row<5>(max_smem);
}

cudaError_t mma_launch(const MmaCall &c, int nsm, cudaStream_t st, int *info) {
    const int L = c.Lb + c.Lk, nhb = nherm(c.Lb);
    const int nnt_total = (c.ncd + 7) / 8;
    const int npass = (nnt_total + NWMAX - 1) / NWMAX;
    const int NW = (nnt_total + npass - 1) / npass;
    const int rs = (nherm(L) + 1) / 2 * 2 + (L > 0 ? (nherm(L - 1) + 1) / 2 * 2 : 2);   // doubles per resident tensor

    // Candidate row-block shapes: one per MW.  cost = warp-steps of GEMM1 per pass (8 m-tiles run abreast),
    // smem decides how many CTAs share an SM.
    struct Cand { int MW, nkb, np, cached, rslots, nblocks, warps; long long cost; size_t smem; int ctas; };
    Cand best{};
    bool have = false;
    // CTA size by measurement: four CTAs of 4 warps per SM for the smaller classes ((ff|ff) 5.5 -> 4.6 ms per 20,000,
    // (fd|dp) 3.7 -> 2.6 ms per 50,000), two CTAs of 8 warps for the large ones ((gg|gg), (ii|ii), (fg|hi) lose 10-40 %
    // with 4 warps); then the row-block shape.
    const bool small = nhb <= 128 && c.ncd <= 64;
    for (int MD_MMA_WARPS = small ? 4 : 8; MD_MMA_WARPS <= 8 && !have; MD_MMA_WARPS += 4)
    for (int MW = 1; MW <= MWMAX; ++MW)
    for (int shrink = 1; shrink <= 256; shrink *= 2) {          // halve the bra primitives per row block until it fits
        const int cap = 8 * MD_MMA_WARPS * MW;
        if (shrink > 1 && (nhb > cap || shrink > c.Kbra)) break;
        Cand k{};
        k.MW = MW;
        if (nhb > cap) {
            const int nblk = (nhb + cap - 1) / cap;
            k.nkb = 1;
            k.np = std::min(cap, ((nhb + nblk - 1) / nblk + 7) / 8 * 8);
            const int nb = (nhb + k.np - 1) / k.np;
            k.nblocks = nb * c.Kbra;
            k.cost = 0;
            for (int b = 0; b < nb; ++b) {
                const int rows = std::min(k.np, nhb - b * k.np);
                k.cost += ((rows + 7) / 8 + MD_MMA_WARPS - 1) / MD_MMA_WARPS;
            }
            k.cost *= c.Kbra;
        } else {
            const int fit = std::max(1, std::min(c.Kbra, cap / nhb) / shrink);
            const int nblk = (c.Kbra + fit - 1) / fit;
            k.nkb = (c.Kbra + nblk - 1) / nblk;
            k.np = nhb;
            k.nblocks = nblk;
            k.cost = 0;
            for (int b = 0; b < nblk; ++b) {
                const int rows = std::min(k.nkb, c.Kbra - b * k.nkb) * nhb;
                k.cost += ((rows + 7) / 8 + MD_MMA_WARPS - 1) / MD_MMA_WARPS;
            }
        }
        // tensors resident in shared memory: all of them when that is cheap, else a batch per row-block
        const size_t budget_all = 72 * 1024;
        const long long nall = (long long)c.Kbra * c.Kket;
        if ((size_t)nall * rs * 8 <= budget_all) { k.cached = 1; k.rslots = (int)nall; }
        else {
            k.cached = 0;
            const int per = std::max<long long>(1, (long long)(48 * 1024) / ((long long)rs * 8 * k.nkb));
            k.rslots = k.nkb * (int)std::min<long long>(per, c.Kket);
        }
        const MmaSmem lay = mma_smem_layout(L, k.rslots, c.Kbra, c.Kket, 8 * MD_MMA_WARPS * MW, 8 * NW + 4);
        k.smem = (size_t)lay.total * 8;
        if (k.smem > (size_t)g_max_smem - 1024) continue;
        k.warps = MD_MMA_WARPS;
        k.ctas = (int)std::max<size_t>(1, std::min<size_t>(16 / MD_MMA_WARPS, (size_t)(g_max_smem + 1024) / (k.smem + 1024)));   // by shared memory and registers
        if (MD_MMA_WARPS == 4 && k.ctas < 4) continue;
        // prefer two CTAs per SM unless one CTA saves more than a third of the warp-steps
        auto score = [](const Cand &x) { return (double)x.cost * (x.ctas >= 2 ? 1.0 : 1.35); };
        // ties: fewer row blocks (each B fragment is reused by more row tiles), then the smaller tile
        const double d = score(k) - score(best);
        if (!have || d < -1e-9 || (d <= 1e-9 && k.nblocks < best.nblocks)) { best = k; have = true; }
    }
    if (!have) return cudaErrorInvalidConfiguration;

    MmaArgs g;
    g.rec_bra = c.rec_bra; g.rec_ket = c.rec_ket; g.stride_bra = c.stride_bra; g.stride_ket = c.stride_ket;
    g.Kbra = c.Kbra; g.Kket = c.Kket; g.Lb = c.Lb; g.Lk = c.Lk; g.nab = c.nab; g.ncd = c.ncd; g.kq0 = c.kq0;
    g.rslots = best.rslots; g.cached = best.cached; g.blk_nkb = best.nkb; g.blk_np = best.np;
    g.qidx = c.qidx; g.nq = c.nq; g.nket = c.nket; g.out = c.out;
    g.s_q = c.s_q; g.s_bi = c.s_bi; g.s_ki = c.s_ki; g.s_ab = c.s_ab; g.s_cd = c.s_cd;
    g.boys_tab = c.boys_tab; g.rlut = c.rlut;
    const unsigned grid = (unsigned)std::min<long long>(c.nq, (long long)nsm * best.ctas);
    g_fn[best.warps == 8][best.MW][NW]<<<grid, 32 * best.warps, best.smem, st>>>(g);
    if (info) {
        info[0] = best.MW; info[1] = NW; info[2] = (int)best.smem; info[3] = best.cached; info[4] = best.rslots;
        info[5] = best.nkb; info[6] = best.np; info[7] = best.ctas;
    }
    return cudaGetLastError();
}

}  // namespace mdb
