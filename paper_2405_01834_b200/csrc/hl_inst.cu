// hl_inst.cu -- host side of the high-l quartet kernel: tile selection, shared-memory carve-up, launch.
#include <algorithm>
#include <cstdio>
#include <cstdlib>

#include "hl_api.cuh"
#include "hl_reg.cuh"

namespace mdb {

namespace {
HlFn g_hl[2][5][5];                   // [0]: 4 warps, [1]: 8 warps; [MW][NW]
HlPairFn g_hl_pair[5];                // [NW]
int g_hl_max_smem = 227 * 1024;
}  // namespace
HlFn *hl_table() { return &g_hl[0][0][0]; }
HlPairFn *hl_pair_table() { return g_hl_pair; }

cudaError_t hl_init(int max_smem, const uint32_t *herm, const double *solid) {
    g_hl_max_smem = max_smem;
    cudaError_t e;
    if ((e = hl_register_w4(max_smem, herm, solid)) != cudaSuccess) return e;
    return hl_register_w8(max_smem, herm, solid);
}

namespace {

struct HlPlan {
    HlArgs a;
    int MW, NW, warps, ctas, npass;
    size_t smem, scratch_bytes;
    unsigned grid;
    int mode;                             // 0 fused (S1 in the quartet kernel), 1 records per shell pair, 2 records per quartet, in chunks
    long long chunk;                      // quartets per launch (mode 2)
    long long recb, reck;                 // doubles per record
    HlPairArgs pb, pk;
    size_t pair_smem_b, pair_smem_k;
};

inline int even_up(int x) { return x + (x & 1); }
inline int up16(int x) { return (x + 15) / 16 * 16; }

// Model cost of the two contractions for one orientation (Table I, columns 3 and 4, per primitive quartet / bra primitive).
double hl_cost(int nhb, int nhk, int nab, int ncd, int Kbra, int Kket) {
    return (double)Kbra * Kket * 2.0 * nhb * nhk * ncd + (double)Kbra * 2.0 * nab * nhb * ncd;
}

bool make_plan(const HlCall &c0, int nsm, HlPlan &P) {
    HlArgs &a = P.a;
    // (ab|cd) = (cd|ab): the side with the cheaper contraction order becomes the kernel's bra (PAPER.md:133, 187 orders the
    // sides for the same reason).  By measurement (profiles/r02_hl_swap.md): whenever the ket has the higher total angular
    // momentum (1.02-1.18x on all ten pairs of orientations tried; the Table-I cost ratio predicts the sign but not the size).
    HlCall c = c0;
    a.qswap = 0;
    {
        const int pure = c0.pure;
        auto sz = [&](const PairView &p, int &nh, int &n, int &K) {
            const int l1 = p.a.l, l2 = p.single ? 0 : p.b.l;
            nh = nherm(l1 + l2); n = ncomp(l1, pure) * ncomp(l2, pure); K = p.a.K * (p.single ? 1 : p.b.K);
        };
        int nhb, nab, Kb, nhk, ncd, Kk;
        sz(c0.bra, nhb, nab, Kb); sz(c0.ket, nhk, ncd, Kk);
        int mode = -1;
        if (const char *f = getenv("MD_HL_SWAP")) mode = atoi(f);
        (void)hl_cost;
        const bool want = mode >= 0 ? mode != 0 : nhk > nhb;          // the side with the higher total l becomes the bra
        if (want && !c0.ket.single && !c0.bra.single) {
            std::swap(c.bra, c.ket);
            std::swap(c.s_bi, c.s_ki); std::swap(c.s_ab, c.s_cd);
            a.qswap = 1;
        }
    }
    a.bra = c.bra; a.ket = c.ket; a.pure = c.pure;
    a.la = c.bra.a.l; a.lb = c.bra.single ? 0 : c.bra.b.l; a.lc = c.ket.a.l; a.ld = c.ket.single ? 0 : c.ket.b.l;
    a.Ka = c.bra.a.K; a.Kb = c.bra.single ? 1 : c.bra.b.K; a.Kc = c.ket.a.K; a.Kd = c.ket.single ? 1 : c.ket.b.K;
    a.Kbra = a.Ka * a.Kb; a.Kket = a.Kc * a.Kd;
    a.Lb = a.la + a.lb; a.Lk = a.lc + a.ld;
    a.nab = ncomp(a.la, c.pure) * ncomp(a.lb, c.pure); a.ncd = ncomp(a.lc, c.pure) * ncomp(a.ld, c.pure);
    a.nhb = nherm(a.Lb); a.nhk = nherm(a.Lk);
    a.nhk_pad = (a.nhk + MD_HL_KC1 - 1) / MD_HL_KC1 * MD_HL_KC1;
    const int nmt2 = (a.nab + 7) / 8;
    int nmt = (a.Kbra * a.nhb + 7) / 8;                   // row tiles if all bra primitives share one row block (refined below)
    a.sb = (8 * nmt2 - 4 + 15) / 16 * 16 + 4;
    a.q_first = (c.ket.single && c.pure) ? nherm(a.lc - 1) / MD_HL_KC1 * MD_HL_KC1 : 0;
    a.qidx = c.qidx; a.nq = c.nq; a.nket = c0.ket.npairs; a.out = c.out;
    a.s_q = c.s_q; a.s_bi = c.s_bi; a.s_ki = c.s_ki; a.s_ab = c.s_ab; a.s_cd = c.s_cd;
    a.boys_tab = c.boys_tab; a.rlut = c.rlut;
    const int L = a.Lb + a.Lk, nR = a.Kbra * a.Kket;
    a.rs0 = even_up(nherm(L)); a.rs1 = even_up(L > 0 ? nherm(L - 1) : 1);

    // cd tile width: as few tiles as possible, at most 4 column tiles of 8 per warp
    const int nnt_total = (a.ncd + 7) / 8;
    const int ntile = (nnt_total + 3) / 4;
    int NW = (nnt_total + ntile - 1) / ntile;
    int warps, MW;
    // By measurement (profiles/r02_autotune.csv, hl rows): 4-warp CTAs (three per SM) for the small classes, else 8 warps; the row tiles
    // per warp that give the fewest tile slots over all row passes, weighted towards larger tiles (fewer gathers per DMMA).
    warps = (nmt <= 12 && nmt2 <= 4 * MD_HL_MT2) ? 4 : 8;
    MW = 1;
    double best = 1e30;
    for (int m = 1; m <= (warps == 4 ? 3 : 4); ++m) {     // critical path in row-tile passes (a ragged last pass only costs the
        double cost = 0;                                   // tiles it has), weighted by the operand traffic per tensor-core step
        for (int left = nmt; left > 0; left -= warps * m) {
            const int t = (std::min(left, warps * m) + warps - 1) / warps;
            cost += t * (1.0 + 0.35 / t);
        }
        if (cost <= best) { best = cost; MW = m; }
    }
    if (const char *f = getenv("MD_HL_FORCE")) {           // measurement override: "MW,NW,warps"
        int m, n, w;
        if (sscanf(f, "%d,%d,%d", &m, &n, &w) == 3 && (w == 4 || w == 8) && m >= 1 && m <= (w == 4 ? 3 : 4) && n >= 1 && n <= 4) {
            MW = m; NW = n; warps = w;
        }
    }
    if (nmt2 > warps * MD_HL_MT2) return false;            // the [ab|cd] tile must fit the GEMM2 accumulators
    const int NT = 8 * NW, NTS = NT + 4;
    a.ntile = (a.ncd + NT - 1) / NT;
    P.MW = MW; P.NW = NW; P.warps = warps;

    const int esz_b = (a.la + 1) * (a.lb + 1) * (a.Lb + 1), esz_k = (a.lc + 1) * (a.ld + 1) * (a.Lk + 1);
    auto t1_slice = [](int l) { const int nc = ncart(l); return (nc >= 21 ? 1 : nc >= 10 ? 2 : nc >= 6 ? 4 : 8) * nc * 20; };   // hl_build_H
    const int t1_b = c.pure ? t1_slice(a.la) : 0, t1_k = c.pure ? t1_slice(a.lc) : 0;
    const int s1_need = std::max(3 * esz_b + 2 + warps * t1_b, 3 * esz_k + 2 + warps * t1_k);
    bool fits = false;
    // bra primitives per row block: all of them if [p~|cd] fits shared memory, else as many as do; then 16 stacked rows
    // per GEMM2 chunk when shared memory allows, else 8
    for (int nblk = 1; nblk <= a.Kbra && !fits; ++nblk)
    for (int kc2 = 16; kc2 >= 8 && !fits; kc2 -= 8) {
        a.kbb = (a.Kbra + nblk - 1) / nblk;
        a.nblk = (a.Kbra + a.kbb - 1) / a.kbb;
        a.mrows = a.kbb * a.nhb;
        a.kc2 = kc2;
        a.mrows_pad = (a.mrows + kc2 - 1) / kc2 * kc2;
        a.ring_stage = up16(std::max(MD_HL_KC1 * NTS, kc2 * a.sb));
        int ov = std::max(a.mrows_pad * NTS, nR * a.rs1);
        ov = std::max(ov, s1_need - MD_HL_STAGES * a.ring_stage);
        a.ov_doubles = up16(ov);
        int o = 0;
        a.o_herm = o; o += even_up(nherm(std::max(a.Lb, a.Lk))) / 2 + 1;
        a.o_rowinfo = o; o += a.mrows_pad;
        a.o_ct = o; o += 4 * 28 * MD_HL_CSTR;
        a.o_hdr = o; o += 4 * (a.Kbra + a.Kket);
        a.o_bar = o; o += 2 * MD_HL_STAGES;
        a.o_r0 = o; o += nR * a.rs0;
        a.o_g0 = o; o += even_up(nR * (L + 1));
        a.o_pq = o; o += even_up(nR * 3);
        o = up16(o);
        a.o_ov = o; o += a.ov_doubles;
        a.o_ring = o; o += MD_HL_STAGES * a.ring_stage;
        o += 128;                                          // fragment loads of row tiles past the end stay inside the allocation
        a.total = o;
        P.smem = (size_t)o * 8;
        fits = P.smem <= (size_t)g_hl_max_smem;
    }
    if (!fits) return false;
    P.npass = (a.mrows_pad / 8 + warps * MW - 1) / (warps * MW);
    if (!hl_table()[((warps == 8) * 5 + MW) * 5 + NW]) return false;

    const long long hb_doubles = (long long)a.nblk * a.mrows_pad * a.sb;
    const long long hk_doubles = (long long)a.ntile * a.Kket * a.nhk_pad * NTS;
    a.off_hk = (hb_doubles + 15) / 16 * 16;
    a.scratch_stride = (a.off_hk + hk_doubles + 15) / 16 * 16;
    P.recb = a.off_hk; P.reck = (hk_doubles + 15) / 16 * 16;
    const int by_regs = warps == 4 ? 3 : 1;             // __launch_bounds__ of hl_kernel
    P.ctas = (int)std::max<size_t>(1, std::min<size_t>(by_regs, (size_t)(g_hl_max_smem + 1024) / (P.smem + 1024)));
    P.grid = (unsigned)std::min<long long>(c.nq, (long long)nsm * P.ctas);

    // Where S1 runs: per shell pair when the pair records fit the budget and pairs are shared by
    // quartets; else per quartet side, in chunks of quartets that fit the budget; else inside the quartet kernel.
    size_t budget = (size_t)2048 << 20;
    if (const char *f = getenv("MD_HL_WS_MB")) budget = (size_t)atoll(f) << 20;
    int mode = -1;
    if (const char *f = getenv("MD_HL_MODE")) mode = atoi(f);
    const long long npb = c.bra.npairs, npk = c.ket.npairs;
    const size_t per_pair = 8 * ((size_t)npb * (P.recb + 4 * a.Kbra) + (size_t)npk * (P.reck + 4 * a.Kket));
    const size_t per_quartet = 8 * (size_t)(P.recb + P.reck + 4 * (a.Kbra + a.Kket));
    if (mode < 0)   // by measurement: records pay when pairs are shared (two quartets per pair or more); else S1 in the kernel
        mode = (per_pair <= budget && npb + npk <= c.nq) ? 1 : 0;
    if (mode == 1 && per_pair > budget) mode = 2;
    if (mode == 2 && per_quartet * P.grid > budget) mode = 0;
    P.mode = mode;
    a.fused = mode == 0; a.by_quartet = mode == 2;
    a.rec_stride_b = P.recb; a.rec_stride_k = P.reck;
    P.chunk = c.nq;
    if (mode == 0) P.scratch_bytes = (size_t)P.grid * a.scratch_stride * 8;
    else if (mode == 1) P.scratch_bytes = per_pair;
    else {
        P.chunk = std::min<long long>(c.nq, (long long)(budget / per_quartet) / P.grid * P.grid);
        P.scratch_bytes = (size_t)P.chunk * per_quartet;
    }
    for (int side = 0; side < 2 && mode; ++side) {
        HlPairArgs &g = side ? P.pk : P.pb;
        g.pv = side ? c.ket : c.bra; g.ket = side;
        g.l1 = side ? a.lc : a.la; g.l2 = side ? a.ld : a.lb; g.K1 = side ? a.Kc : a.Ka; g.K2 = side ? a.Kd : a.Kb;
        g.pure = c.pure; g.nh = side ? a.nhk : a.nhb; g.nh_pad = side ? a.nhk_pad : 0; g.sb = side ? 0 : a.sb;
        g.tile_stride = side ? (long long)a.Kket * a.nhk_pad * NTS : 0;
        g.kbb = side ? 1 : a.kbb; g.blk_rows = side ? 0 : a.mrows_pad;
        g.rec_stride = side ? P.reck : P.recb;
        g.by_quartet = mode == 2; g.qidx = c.qidx; g.nket = c0.ket.npairs; g.qswap = a.qswap;
        const int esz = (g.l1 + 1) * (g.l2 + 1) * (g.l1 + g.l2 + 1);
        int o = 0;
        g.o_herm = o; o += nherm(g.l1 + g.l2) / 2 + 1;
        g.o_ct = o; o += 4 * 28 * MD_HL_CSTR;
        o = up16(o);
        g.o_ws = o;
        g.ws_doubles = 3 * esz + 2 + (c.pure ? 4 * t1_slice(g.l1) : 0);                      // 4 warps (hl_pair_kernel)
        o += g.ws_doubles;
        (side ? P.pair_smem_k : P.pair_smem_b) = (size_t)o * 8;
    }
    return true;
}

}  // namespace

int hl_plan(const HlCall &c, int nsm, size_t *scratch_bytes) {
    HlPlan P;
    if (!make_plan(c, nsm, P)) return 0;
    *scratch_bytes = P.scratch_bytes;
    return 1;
}

cudaError_t hl_launch(const HlCall &c, int nsm, void *scratch, cudaStream_t st, int *info, int *launches) {
    HlPlan P;
    if (!make_plan(c, nsm, P)) return cudaErrorInvalidConfiguration;
    HlFn fn = hl_table()[((P.warps == 8) * 5 + P.MW) * 5 + P.NW];
    HlArgs &a = P.a;
    *launches = 0;
    if (P.mode == 0) {
        a.scratch = (double *)scratch;
        a.q_begin = 0; a.q_end = c.nq;
        fn<<<P.grid, 32 * P.warps, P.smem, st>>>(a);
        ++*launches;
    } else {
        // record layout in the workspace: [bra records][ket records][bra headers][ket headers]; padding stays zero
        cudaError_t e = cudaMemsetAsync(scratch, 0, P.scratch_bytes, st);
        if (e != cudaSuccess) return e;
        const long long nrb = P.mode == 1 ? P.pb.pv.npairs : P.chunk, nrk = P.mode == 1 ? P.pk.pv.npairs : P.chunk;   // kernel's sides (maybe swapped)
        double *recb = (double *)scratch, *reck = recb + nrb * P.recb;
        double *hdrb = reck + nrk * P.reck, *hdrk = hdrb + nrb * 4 * a.Kbra;
        a.rec_b = recb; a.rec_k = reck; a.hdr_b = hdrb; a.hdr_k = hdrk;
        P.pb.rec = recb; P.pb.hdr = hdrb; P.pk.rec = reck; P.pk.hdr = hdrk;
        HlPairFn pfn = hl_pair_table()[P.NW];
        for (long long q0 = 0; q0 < c.nq; q0 += P.chunk) {
            const long long q1 = std::min(c.nq, q0 + P.chunk);
            if (P.mode == 2 || q0 == 0) {
                P.pb.nrec = P.mode == 1 ? nrb : q1 - q0; P.pk.nrec = P.mode == 1 ? nrk : q1 - q0;
                P.pb.q_begin = P.pk.q_begin = q0;
                const unsigned gb = (unsigned)std::min<long long>(P.pb.nrec, (long long)nsm * 4);
                const unsigned gk = (unsigned)std::min<long long>(P.pk.nrec, (long long)nsm * 4);
                if (gb) { pfn<<<gb, 128, P.pair_smem_b, st>>>(P.pb); ++*launches; }
                if (gk) { pfn<<<gk, 128, P.pair_smem_k, st>>>(P.pk); ++*launches; }
            }
            a.q_begin = q0; a.q_end = q1;
            const unsigned grid = (unsigned)std::min<long long>(q1 - q0, (long long)P.grid);
            fn<<<grid, 32 * P.warps, P.smem, st>>>(a);
            ++*launches;
        }
    }
    if (info) {
        info[0] = P.MW; info[1] = P.NW; info[2] = P.warps; info[3] = (int)P.smem; info[4] = P.ctas; info[5] = P.npass;
        info[6] = P.mode; info[7] = (int)P.grid;
    }
    return cudaGetLastError();
}

}  // namespace mdb
