// fused2_main.cuh -- the kernel body of the warp-specialised fused kernel (see fused2_kernel.cuh).
#pragma once
#include <cuda_pipeline.h>

#include "fused2_kernel.cuh"

namespace mdb {

struct Fused2Args {
    FusedArgs f;                  // shells, index lists, output strides (as for fused_kernel)
    double *scratch;              // per-CTA pair-table scratch (stays in L2): [grid][NQ][Kbra*TB + Kket*TK]
    int NQ;                       // quartets per CTA pass
    int TCH;                      // consumer threads per cd chunk (multiple of 32, >= NQ*NPG)
};

// P4 for one batch and one cd chunk CH: hacc[k][comp] += E[e] * R[p_k + q(e)]   (Eq. 25).
// Software-pipelined by hand: the E pairs are loaded ED pairs ahead and the Hermite integrals of a q~
// group RD groups ahead of their use, into register rings indexed by compile-time constants, so that
// the ~30-cycle shared-memory latency is covered inside one warp (there are only 1-2 consumer warps per
// scheduler).
template <class C, int LC, int LD, int PB, int NCH, int CH>
__device__ __forceinline__ void f2_contract(double (&hacc)[PB][C::NACC], const double *Rb, const int (&pofs)[PB],
                                            const double *EP) {
    using QGT = QGroups<LC, LD, NCH, CH>;
    constexpr ProdQ<LC, LD, NCH> PQ{};
    constexpr int E0 = PQ.choff[CH], NE = PQ.choff[CH + 1] - E0, NPAIR = NE / 2;
    constexpr int NG = QGT{}.ng;
    constexpr int ED = 4, RD = 2;
    const double2 *ep2 = (const double2 *)(EP + E0);
    double2 eb[ED + 1];
    double rb[RD + 1][PB];
    auto loadR = [&](auto sc) {
        constexpr int s = decltype(sc)::value;
        constexpr XYZ h = herm_exp(QGT{}.gq[s]);
        constexpr int qo = C::BR.A * h.x + C::BR.B * h.y + h.z;          // index(p~+q~) = index(p~) + index(q~)
#pragma unroll
        for (int k = 0; k < PB; ++k) rb[s % (RD + 1)][k] = Rb[pofs[k] + qo];
    };
    static_for<(RD < NG ? RD : NG)>([&](auto sc) { loadR(sc); });
    static_for<(ED < NPAIR ? ED : NPAIR)>([&](auto pc) { eb[decltype(pc)::value % (ED + 1)] = ep2[decltype(pc)::value]; });
    static_for<NE>([&](auto ec) {
        constexpr int e = decltype(ec)::value;
        constexpr int s = QGT{}.gid[e];
        if constexpr ((e & 1) == 0 && e / 2 + ED < NPAIR) eb[(e / 2 + ED) % (ED + 1)] = ep2[e / 2 + ED];
        if constexpr (s >= 0) {
            constexpr bool starts = QGT{}.gs[s] == e && s + RD < NG;
            if constexpr (starts) loadR(std::integral_constant<int, s + RD>{});
            constexpr int comp = PQ.comp_of[E0 + e];
            const double2 &p2 = eb[(e / 2) % (ED + 1)];
            const double x = (e & 1) ? p2.y : p2.x;
#pragma unroll
            for (int k = 0; k < PB; ++k) hacc[k][comp] = fma(x, rb[s % (RD + 1)][k], hacc[k][comp]);
        }
    });
}

// One product-list entry from a table record and its packed word (fused2_tables.cuh).
__device__ __forceinline__ double prod_entry(const double *tab, unsigned w) {
    return (tab[w & 255] * tab[w >> 8 & 255]) * (tab[w >> 16 & 255] * tab[w >> 24]);
}

// Store to the per-CTA scratch with an L2 evict_last policy: the scratch is rewritten for every group of
// quartets and re-read once per bra primitive, so it should stay in L2 and never reach DRAM.
__device__ __forceinline__ void st_scratch(double *p, double v) {
    unsigned long long pol;
    asm volatile("createpolicy.fractional.L2::evict_last.b64 %0, 1.0;" : "=l"(pol));
    asm volatile("st.global.L2::cache_hint.f64 [%0], %1, %2;" ::"l"(p), "d"(v), "l"(pol) : "memory");
}

// n products of one table record, entries w, w + stride, ...: written to the scratch; all loads of a
// batch of four entries are issued before the first store.
__device__ __forceinline__ void prod_list(const double *tab, const unsigned *pack, double *dst, int n, int w, int stride) {
    for (int e0 = w; e0 < n; e0 += 4 * stride) {
        unsigned ww[4];
        double v[4];
#pragma unroll
        for (int u = 0; u < 4; ++u) ww[u] = e0 + u * stride < n ? pack[e0 + u * stride] : PROD_WORD_ZERO;
#pragma unroll
        for (int u = 0; u < 4; ++u) v[u] = prod_entry(tab, ww[u]);
#pragma unroll
        for (int u = 0; u < 4; ++u)
            if (e0 + u * stride < n) st_scratch(dst + e0 + u * stride, v[u]);
    }
}

// Copy n doubles global -> shared, eight loads in flight per thread.
__device__ __forceinline__ void copy_in(double *dst, const double *src, int n, int t, int nt) {
    for (int i0 = t; i0 < n; i0 += 8 * nt) {
        double v[8];
#pragma unroll
        for (int u = 0; u < 8; ++u) v[u] = i0 + u * nt < n ? __ldcg(src + i0 + u * nt) : 0.0;
#pragma unroll
        for (int u = 0; u < 8; ++u)
            if (i0 + u * nt < n) dst[i0 + u * nt] = v[u];
    }
}

// Flush of one chunk of a consumer thread's [p~|cd] accumulators to the drain rows half[p~][cd_out].
// Cartesian output: the chunk's own columns.  Solid output: both ket transforms (Eq. 16) in registers -- the d
// index fully, the c index over the chunk's components only -- so the row receives a partial sum; chunk 0
// stores, later chunks add (ADD), in chunk order, with a consumer barrier between the rounds.
template <class C, int LC, int LD, bool PURE, int PB, bool ADD>
__device__ __forceinline__ void f2_flush(const double (&hacc)[PB][C::NACC], int c0, const int (&ip)[PB], double *half) {
#pragma unroll
    for (int k = 0; k < PB; ++k) {
        if (ip[k] < 0) continue;
        double *row = half + ip[k] * C::HS;
        if constexpr (!PURE) {
#pragma unroll
            for (int cl = 0; cl < C::CHC; ++cl) {
                if (c0 + cl >= C::NCC) break;
#pragma unroll
                for (int d = 0; d < C::NCD; ++d) row[(c0 + cl) * C::NCD + d] = hacc[k][cl * C::NCD + d];
            }
        } else {
            constexpr SolidTab<LD> SD{};
            constexpr SolidTab<LC> SC{};
            double t[C::CHC][C::NDO];                        // d index transformed
#pragma unroll
            for (int cl = 0; cl < C::CHC; ++cl)
#pragma unroll
                for (int m = 0; m < C::NDO; ++m) {
                    double s = 0.0;
#pragma unroll
                    for (int d = 0; d < C::NCD; ++d)
                        if (SD.c[m][d] != 0.0) s = fma(SD.c[m][d], hacc[k][cl * C::NCD + d], s);
                    t[cl][m] = s;
                }
            // c index: the chunk is known only at run time, the coefficients come from a small constant table
#pragma unroll
            for (int mc = 0; mc < C::NCO; ++mc)
#pragma unroll
                for (int m = 0; m < C::NDO; ++m) {
                    double s = ADD ? row[mc * C::NDO + m] : 0.0;
#pragma unroll
                    for (int cl = 0; cl < C::CHC; ++cl)
                        if (c0 + cl < C::NCC) s = fma(d_solidc<LC>.c[mc][c0 + cl], t[cl][m], s);
                    row[mc * C::NDO + m] = s;
                }
            (void)SC;
        }
    }
}

template <int LA, int LB, int LC, int LD, bool PURE, int PB, int NCH>
__global__ void __launch_bounds__(MD_F2_PRODUCERS + 192, 1) fused2_kernel(Fused2Args ga) {
    using C = F2Cfg<LA, LB, LC, LD, PURE, PB, NCH>;
    using I = F2Impl<LA, LB, LC, LD, PURE, PB, NCH>;
    constexpr int L = C::L;
    const FusedArgs &g = ga.f;
    extern __shared__ double sm[];
    const int NQ = ga.NQ, NC = NCH * ga.TCH, NT = blockDim.x, NP = NT - NC, NG = NP / 2;
    // carve-up: [NQ] x { sidx[4 ints], output base, pad }, [NQ] x NBUF consumer buffers, 2 x [NQ] producer-group
    // scratch, packed product words.  The drain region {[p~|c md] rows, bra products} of a quartet aliases the
    // two buffers of the producer group that built the last batch of the bra primitive.
    double *perq = sm;
    double *bufs = sm + (size_t)NQ * C::PERQ;
    double *gsc = bufs + (size_t)NQ * C::CBQ;
    unsigned *packq = (unsigned *)(gsc + (size_t)2 * NQ * C::GS);          // [EPK]  ket product words
    unsigned *packc = packq + even_up(C::EPK);                             // [NPB]  bra product words
    double *epb = gsc + (size_t)2 * NQ * C::GS + C::FIXED;                 // [NQ][EPBS] head of the bra product list being drained
    constexpr int O_OB = 2;
    constexpr int EPKe = even_up(C::EPK), NPBe = even_up(C::NPB);
    constexpr int KREC = 8 + EPKe, BRECS = 8 + NPBe;                       // scratch records: header + product list
    auto cbuf = [&](int b, int j) { return bufs + (size_t)j * C::CBQ + b * C::CB; };
    const int tid = threadIdx.x;
    const bool consumer = tid < NC;
    const int ptid = tid - NC;
    const int Ka = g.bra.a.K, Kb = g.bra.single ? 1 : g.bra.b.K;
    const int Kc = g.ket.a.K, Kd = g.ket.single ? 1 : g.ket.b.K;
    const int Kbra = Ka * Kb, Kket = Kc * Kd, B = Kbra * Kket;             // B batches per group of quartets
    const size_t SCRQ = (size_t)Kbra * BRECS + (size_t)Kket * KREC;        // scratch doubles per quartet
    double *scr = ga.scratch + (size_t)blockIdx.x * NQ * SCRQ;
    auto scr_bra = [&](int j, int kb) { return scr + (size_t)j * SCRQ + (size_t)kb * BRECS; };
    auto scr_ket = [&](int j, int kk) { return scr + (size_t)j * SCRQ + (size_t)Kbra * BRECS + (size_t)kk * KREC; };
    // batch b = kb*Kket + kk is built by producer group b&1 in that group's buffer slot (b>>1)&1
    auto buf_of = [](int b) { return (b & 1) * 2 + (b >> 1 & 1); };
    auto is_last = [&](int b) { return b < B && b % Kket == Kket - 1; };   // last batch of its bra primitive
    // buffers that become a drain region are released by the drain's last barrier, not by the EMPTY handshake
    auto deferred = [&](int b) { return is_last(b) || is_last(b + 2); };

    // consumer role: chunk ch, quartet slot cj, Hermite rows ip[k]
    int ch = 0, cj = 0, ip[PB], pofs[PB];
    bool cact = false;
    if (consumer) {
        ch = tid / ga.TCH;
        const int r = tid - ch * ga.TCH;
        cact = r < NQ * C::NPG;
        cj = r / C::NPG;
        const int pg = r - cj * C::NPG;
#pragma unroll
        for (int k = 0; k < PB; ++k) {
            const int i = d_pmap<C::Lb, PB, L>.p[k][pg];
            ip[k] = cact ? i : -1;
            // a lane without a row in this slot reads its neighbour's address (same half-warp: a broadcast)
            const int in = i < 0 ? d_pmap<C::Lb, PB, L>.p[k][(pg ^ 1) < C::NPG ? (pg ^ 1) : 0] : i;
            const int w = d_herm<C::NHB>.e[in < 0 ? 0 : in];
            pofs[k] = C::BR.A * (w & 0xff) + C::BR.B * (w >> 8 & 0xff) + (w >> 16);
        }
    }
    for (int e = tid; e < C::EPK; e += NT) packq[e] = d_packq<LC, LD, NCH>.w[e];
    for (int e = tid; e < C::NPB; e += NT) packc[e] = d_packc<LA, LB>.w[e];
    if (tid < EPKe - C::EPK) packq[C::EPK + tid] = PROD_WORD_ZERO;
    if (tid < NPBe - C::NPB) packc[C::NPB + tid] = PROD_WORD_ZERO;

    const long long ngroups = (g.nq + NQ - 1) / NQ;
    for (long long grp = blockIdx.x; grp < ngroups; grp += gridDim.x) {
        const long long q0 = grp * NQ;
        const int nqg = (int)min((long long)NQ, g.nq - q0);
        __syncthreads();                                     // previous group is done with shared memory
        if (tid < nqg) {
            const long long q = q0 + tid;
            long long bi, ki;
            if (g.qidx) { bi = g.qidx[2 * q]; ki = g.qidx[2 * q + 1]; }
            else { bi = q / g.nket; ki = q % g.nket; }
            long long ia = bi, ib = bi, ic = ki, id = ki;
            if (g.bra.idx) { ia = g.bra.idx[2 * bi + g.bra_swap]; ib = g.bra.idx[2 * bi + 1 - g.bra_swap]; }
            if (g.ket.idx) { ic = g.ket.idx[2 * ki + g.ket_swap]; id = g.ket.idx[2 * ki + 1 - g.ket_swap]; }
            double *pq = perq + (size_t)tid * C::PERQ;
            int *sidx = (int *)pq;
            sidx[0] = (int)ia; sidx[1] = (int)ib; sidx[2] = (int)ic; sidx[3] = (int)id;
            *(long long *)(pq + O_OB) = q * g.s_q + bi * g.s_bi + ki * g.s_ki;
        }
        __syncthreads();
        // ---- S1, once per group, by all threads, into this CTA's scratch (global memory that stays in L2): for every
        // bra and every ket primitive pair of these quartets a record {header, product list}: the 1-D tables
        // (Eqs. 9, 10, 13, 14) pass through shared memory (the batch buffers are idle here), a chunk of primitives
        // at a time; the lists E^{ab}_{p~} and E^{cd}_{q~}(-1)^{|q~|} (Eqs. 7, 19) do not depend on the other side.
        auto build_side = [&](auto side) {
            constexpr bool KET = decltype(side)::value;
            constexpr int T = KET ? C::TK : C::TB, LEN = KET ? EPKe : NPBe;
            const int K = KET ? Kket : Kbra, K2 = KET ? Kd : Kb;
            const unsigned *pack = KET ? packq : packc;
            const int KC = min(K, C::CBQ / T);
            for (int k0 = 0; k0 < K; k0 += KC) {
                const int kc = min(KC, K - k0);
                for (int it = tid; it < 3 * nqg * kc; it += NT) {
                    const int ax = it % 3, r = it / 3, j = r / kc, k = r - j * kc;
                    const int *sidx = (const int *)(perq + (size_t)j * C::PERQ);
                    double *tab = bufs + (size_t)j * C::CBQ + (size_t)k * T;
                    if constexpr (KET) table_task<LC, LD>(g.ket, sidx[2], sidx[3], (k0 + k) / K2, (k0 + k) % K2, ax, tab);
                    else table_task<LA, LB>(g.bra, sidx[0], sidx[1], (k0 + k) / K2, (k0 + k) % K2, ax, tab);
                }
                __syncthreads();
                for (int r = tid >> 5; r < nqg * kc; r += NT >> 5) {      // one warp per (quartet, primitive pair)
                    const int j = r / kc, k = r - j * kc;
                    const double *tab = bufs + (size_t)j * C::CBQ + (size_t)k * T;
                    double *rec = KET ? scr_ket(j, k0 + k) : scr_bra(j, k0 + k);
                    if ((tid & 31) < 8) st_scratch(rec + (tid & 31), tab[tid & 31]);
                    prod_list(tab, pack, rec + 8, LEN, tid & 31, 32);
                }
                __syncthreads();
            }
        };
        build_side(std::false_type{});
        build_side(std::true_type{});

        // ---- the drain of bra primitive kb (Eq. 16 on c, Eq. 26, bra transform, output), run by the consumers and the
        // producer group dg whose two buffers hold the drain region; t = 0..DN-1 numbers the participants.
        auto drain_phase = [&](int kb, int dg, int t) {
            const int DN = NC + NG, DB = F2_BAR_DRAIN + dg;
            auto dreg = [&](int j) { return cbuf(2 * dg, j); };
            bar_sync(DB, DN);                                // the [p~|cd] rows are flushed
            // P5: [ab|cd] += sum_p~ E^{ab}_{p~} [p~|cd]  (Eq. 26), bra transform, accumulate in the output (L2)
            for (int it = t; it < nqg * C::NCD_O; it += DN) {
                const int j = it / C::NCD_O, icd = it - j * C::NCD_O;
                const double *half = dreg(j) + C::O_HALF + icd;
                double hv[C::NHB];
#pragma unroll
                for (int i = 0; i < C::NHB; ++i) hv[i] = half[i * C::HS];
                double oacc[C::NAB_C];
#pragma unroll
                for (int i = 0; i < C::NAB_C; ++i) oacc[i] = 0.0;
                const double2 *ep = (const double2 *)(scr_bra(j, kb) + 8);     // tail of the bra product list: L2 scratch through L1
                const double2 *es = (const double2 *)(epb + (size_t)j * C::EPBS);   // its head: staged by the consumers
                constexpr ProdList<LA, LB, 0> PBL{};
                double2 e2 = make_double2(0.0, 0.0);
                static_for<PBL.N>([&](auto ic) {
                    constexpr int i = decltype(ic)::value;
                    if constexpr ((i & 1) == 0) e2 = i < C::EPBS ? es[i / 2] : ep[i / 2];
                    oacc[PBL.comp[i]] = fma((i & 1) ? e2.y : e2.x, hv[PBL.off[i]], oacc[PBL.comp[i]]);
                });
                double o2[C::NAB_O];
                solid2<LA, LB, PURE>(oacc, o2);
                double *o = g.out + *(const long long *)(perq + (size_t)j * C::PERQ + O_OB) + (icd / C::NDO) * g.sc + (icd % C::NDO) * g.sd;
                if (kb > 0) {                                // later bra primitives: reduction in L2, nothing comes back
#pragma unroll
                    for (int a = 0; a < C::NAO; ++a)
#pragma unroll
                        for (int b = 0; b < C::NBO; ++b)
                            asm volatile("red.global.add.f64 [%0], %1;" ::"l"(o + a * g.sa + b * g.sb), "d"(o2[a * C::NBO + b]) : "memory");
                } else {
#pragma unroll
                    for (int a = 0; a < C::NAO; ++a)
#pragma unroll
                        for (int b = 0; b < C::NBO; ++b) o[a * g.sa + b * g.sb] = o2[a * C::NBO + b];
                }
            }
            bar_sync(DB, DN);                                // the drain region is free again
        };

        if (consumer) {
            // ---------------- consumers: P4 over the ket primitives, then the drain ----------------
            for (int kb = 0; kb < Kbra; ++kb) {
                // the previous drain is over for every participant: stage this primitive's bra product list behind P4
                if constexpr (C::EPBS > 0) {
                    constexpr int H = C::EPBS / 2;
                    for (int c = tid; c < nqg * H; c += NC) {
                        const int j = c / H, i = c - j * H;
                        __pipeline_memcpy_async(epb + (size_t)j * C::EPBS + 2 * i, scr_bra(j, kb) + 8 + 2 * i, 16);
                    }
                    __pipeline_commit();
                }
                double hacc[PB][C::NACC];
#pragma unroll
                for (int k = 0; k < PB; ++k)
#pragma unroll
                    for (int i = 0; i < C::NACC; ++i) hacc[k][i] = 0.0;
                for (int kk = 0; kk < Kket; ++kk) {
                    const int b = kb * Kket + kk, buf = buf_of(b);
                    bar_sync(F2_BAR_FULL + buf, NC + NG);
                    if (cact && cj < nqg) {
                        const double *rec = cbuf(buf, cj);
                        const double *Rb = rec + C::O_R;
                        const double *EP = rec + C::O_EP;
                        if (NCH == 1 || ch == 0) f2_contract<C, LC, LD, PB, NCH, 0>(hacc, Rb, pofs, EP);
                        if constexpr (NCH > 1) { if (ch == 1) f2_contract<C, LC, LD, PB, NCH, 1>(hacc, Rb, pofs, EP); }
                        if constexpr (NCH > 2) { if (ch == 2) f2_contract<C, LC, LD, PB, NCH, 2>(hacc, Rb, pofs, EP); }
                    }
                    if (b + 4 < B && !deferred(b)) bar_arrive(F2_BAR_EMPTY + buf, NC + NG);
                }
                const int dg = (kb * Kket + Kket - 1) & 1;
                __pipeline_wait_prior(0);                    // this thread's part of the staged list has landed
                bar_sync(F2_BAR_CONS, NC);                   // every consumer is done with group dg's buffers
                if (cact && cj < nqg && ch == 0)
                    f2_flush<C, LC, LD, PURE, PB, false>(hacc, 0, ip, cbuf(2 * dg, cj) + C::O_HALF);
                if constexpr (PURE && NCH > 1) {             // solid output: later chunks add their partial c transform
#pragma unroll
                    for (int r = 1; r < NCH; ++r) {
                        bar_sync(F2_BAR_CONS, NC);
                        if (cact && cj < nqg && ch == r)
                            f2_flush<C, LC, LD, PURE, PB, true>(hacc, r * C::CHC, ip, cbuf(2 * dg, cj) + C::O_HALF);
                    }
                } else if constexpr (NCH > 1) {
                    if (cact && cj < nqg && ch > 0)
                        f2_flush<C, LC, LD, PURE, PB, false>(hacc, ch * C::CHC, ip, cbuf(2 * dg, cj) + C::O_HALF);
                }
                drain_phase(kb, dg, tid);
            }
        } else {
            // ---------------- producers: Boys, Hermite Coulomb tensors, product-list streaming ----------------
            // Two groups build alternate batches, each in two buffers of its own, and run ahead across bra primitives.
            const int pgp = ptid / NG, gt = ptid - pgp * NG;
            double *gs0 = gsc + (size_t)pgp * NQ * C::GS;
            for (int b = pgp; b < B; b += 2) {
                const int kb = b / Kket, kk = b - kb * Kket, buf = buf_of(b);
                if (b >= 4 && !deferred(b - 4)) bar_sync(F2_BAR_EMPTY + buf, NC + NG);
                // stage 0: the product list of ket primitive kk, L2 -> shared memory by asynchronous 16-byte copies
                // that complete behind the recursion stages
                for (int c = gt; c < nqg * (EPKe / 2); c += NG) {
                    const int j = c / (EPKe / 2), i = c - j * (EPKe / 2);
                    __pipeline_memcpy_async(cbuf(buf, j) + C::O_EP + 2 * i, scr_ket(j, kk) + 8 + 2 * i, 16);
                }
                __pipeline_commit();
                if (gt < nqg)                                             // stage 1: Boys, [0]^(m), z-line
                    I::z_task(scr_bra(gt, kb), scr_ket(gt, kk), gs0 + (size_t)gt * C::GS, cbuf(buf, gt), g.boys_tab);
                bar_sync(F2_BAR_PROD + pgp, NG);
                for (int it = gt; it < (L + 1) * nqg; it += NG) {         // stage y (tasks sorted by line length)
                    const int v = it / nqg, j = it - v * nqg;
                    I::y_task(v, gs0 + (size_t)j * C::GS, cbuf(buf, j));
                }
                bar_sync(F2_BAR_PROD + pgp, NG);
                for (int it = gt; it < C::NZ * nqg; it += NG) {           // stage x (sorted by line length)
                    const int c = it / nqg, j = it - c * nqg;
                    // column u of the anti-diagonal u + v = s: s = floor((sqrt(8c + 1) - 1)/2), exact in float for c < 2^20
                    const int s = (int)((sqrtf((float)(8 * c + 1)) - 1.0f) * 0.5f);
                    const int u = c - ((s * (s + 1)) >> 1);
                    I::x_task(u, s - u, gs0 + (size_t)j * C::GS, cbuf(buf, j));
                }
                __pipeline_wait_prior(0);
                bar_arrive(F2_BAR_FULL + buf, NC + NG);
                if (kk == Kket - 1) drain_phase(kb, pgp, NC + gt);        // this group's buffers become the drain region
            }
        }
    }
}

}  // namespace mdb
