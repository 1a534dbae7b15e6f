// fused2_kernel.cuh -- warp-specialised compile-time-l fused kernel: ONE launch runs S1-S5 of a class
// (la lb|lc ld) with no intermediate in HBM, built for contracted shells.
//
// A CTA holds NC consumer threads and NP producer threads and works on NQ quartets at a time.
// For every bra primitive kb and ket primitive kk (a "batch" = that primitive quartet of all NQ
// quartets) the PRODUCER warps build, in one of two shared-memory buffers,
//   stage 0  the ket 1-D tables E^t_{ij} of primitive kk               (Eqs. 9,10,13,14)
//   stage 1  [0]^(m) (Eqs. 21-23, Boys function) and from it the z-line [00v]^(m);
//            the ket products E^{cd}_{q~}(-1)^{|q~|}, q~-major               (Eqs. 7, 19)
//   stage y  [0uv]^(m) from [00v]^(m)                                         (Eq. 24 on u)
//   stage x  [tuv]^(0) from [0uv]^(m), stored in an additive bank-aware layout   (Eq. 24 on t)
// while the CONSUMER warps contract the other buffer,
//   P4  [p~|cd] += sum_q~ E^{cd}_{q~} [p~+q~]^(0)                              (Eq. 25)
// each thread owning PB Hermite rows p~ and one chunk of cd in REGISTERS for the whole kk loop.
// Eq. 24 is applied one Cartesian direction at a time: a thread that owns a line (all t for fixed
// u,v) needs only the [0uv]^(m), m = 0..L-u-v, of that line and two register rows, so the
// recursion costs three producer-only barriers per batch instead of one CTA barrier per level.
// The two buffers are handed over with named barriers (bar.arrive / bar.sync).
// After the kk loop of a bra primitive the whole CTA transforms the ket to solid harmonics
// (Eq. 16), applies Eq. 26 ([ab|cd] += sum_p~ E^{ab}_{p~} [p~|cd]) with the bra transform, and
// accumulates into the output block, which stays in L2 between bra primitives.
#pragma once
#include <cuda_pipeline.h>
#include "boys.cuh"
#include "fused2_tables.cuh"
#include "fused_kernel.cuh"      // axis_table, solid2, FusedArgs

namespace mdb {

#define MD_F2_PRODUCERS 192          // two groups of three warps

template <int LA, int LB, int LC, int LD, bool PURE, int PB, int NCH>
struct F2Cfg {
    static constexpr int Lb = LA + LB, Lk = LC + LD, L = Lb + Lk;
    static constexpr int NHB = nherm(Lb), NHK = nherm(Lk), NHL = nherm(L);
    static constexpr int NCA = ncart(LA), NCB = ncart(LB), NCC = ncart(LC), NCD = ncart(LD);
    static constexpr int NAO = ncomp(LA, PURE), NBO = ncomp(LB, PURE), NCO = ncomp(LC, PURE), NDO = ncomp(LD, PURE);
    static constexpr int NAB_C = NCA * NCB, NAB_O = NAO * NBO, NCD_O = NCO * NDO;
    static constexpr int NPG = (NHB + PB - 1) / PB;            // p~ groups per quartet
    static constexpr int CHC = (NCC + NCH - 1) / NCH;          // c components per chunk
    static constexpr int NACC = CHC * NCD;                     // accumulators per p~
    static constexpr int E1B = e1_count(LA, LB), E1K = e1_count(LC, LD);
    static constexpr int TB = even_up(8 + 3 * E1B), TK = even_up(8 + 3 * E1K);   // table records
    static constexpr int NPB = ProdCount<LA, LB>::value();
    static constexpr int EPK = ProdQ<LC, LD, NCH>{}.len();
    static constexpr int HW = NCO * NDO;                       // cd_out: both ket transforms are applied before the flush
    static constexpr int HS = HW | 1;                          // odd row stride: conflict-free columns
    static constexpr int NZ = (L + 1) * (L + 2) / 2;           // entries of the z-line output
    static constexpr Brick BR = brick_layout(L, Lb);
    static_assert(brick_injective(L, BR), "brick layout must be injective");
    static constexpr int NRA = even_up(BR.foot > NZ ? BR.foot : NZ);
    // consumer-visible buffer of one quartet and batch (doubles): what P4 reads
    static constexpr int O_R = 0;                              // z-line output, later [r]^(0) in the brick layout
    static constexpr int O_EP = NRA;                           // ket product list
    static constexpr int CB = O_EP + even_up(EPK);
    static constexpr int NBUF = 4;                             // two per producer group
    // producer-group scratch of one quartet: only live while a batch is being built
    static constexpr int O_B = 0;                              // [0uv]^(m) columns
    static constexpr int O_PQ = O_B + even_up(NHL);            // X, Y, Z, pad
    // strides between quartets are 2 mod 4 doubles: lanes that do the same task for 8 consecutive quartets
    // then fall on 8 distinct 8-byte banks
    static constexpr int pad_bank(int x) { return x + ((2 - x) % 4 + 4) % 4; }
    static constexpr int GS = pad_bank(O_PQ + 4);
    static constexpr int CBQ = NBUF * CB + ((10 - NBUF * CB) % 16 + 16) % 16;   // the NBUF buffers of one quartet: 10 (mod 16), see PMap
    // drain region of one quartet, aliased on its NBUF buffers once every batch of the bra primitive is consumed
    static constexpr int O_HALF = 0, O_EPB = even_up(NHB * HS);
    static_assert(O_EPB <= 2 * CB, "the [p~|cd] rows must fit in the two buffers of one producer group");
    // per quartet, never aliased: shell indices, output base
    static constexpr int PERQ = 4;
    static constexpr int QTOT0 = PERQ + CBQ + 2 * GS;
    static constexpr int FIXED = even_up((even_up(EPK) + even_up(NPB)) / 2);   // packed product words (doubles)
    // Bra product list of the bra primitive being drained, staged in shared memory: as many entries per quartet as the
    // shared memory left over at the class's quartet count allows (the rest of the list is read from the L2 scratch).
    static constexpr int SMEM_D = 232448 / 8;                  // 227 KB per CTA on sm_100a, in doubles
    static constexpr int NQCAP = (192 / NCH) / NPG < 64 ? (192 / NCH) / NPG : 64;   // fused2_inst.cu: consumer threads per chunk
    static constexpr int NQ0 = (SMEM_D - FIXED) / QTOT0 < NQCAP ? (SMEM_D - FIXED) / QTOT0 : NQCAP;
    static constexpr int EPBS_ROOM = NQ0 < 1 ? 0 : (((SMEM_D - FIXED) / NQ0 - QTOT0) & ~1);
    static constexpr int EPBS = EPBS_ROOM < 16 ? 0 : (EPBS_ROOM < even_up(NPB) ? EPBS_ROOM : even_up(NPB));
    static constexpr int QTOT = QTOT0 + EPBS;
    static __host__ __device__ constexpr size_t smem_bytes(int nq) { return 8 * ((size_t)nq * QTOT + FIXED); }
};

__device__ __forceinline__ void bar_sync(int id, int n) { asm volatile("bar.sync %0, %1;" ::"r"(id), "r"(n) : "memory"); }
__device__ __forceinline__ void bar_arrive(int id, int n) {
    __threadfence_block();
    asm volatile("bar.arrive %0, %1;" ::"r"(id), "r"(n) : "memory");
}
enum { F2_BAR_PROD = 2, F2_BAR_CONS = 4, F2_BAR_FULL = 5, F2_BAR_EMPTY = 9, F2_BAR_DRAIN = 13 };   // FULL/EMPTY: 4 ids each; PROD, DRAIN: 2

// One axis of the two-centre table, written compactly (rows (i,j), t = 0..i+j).
template <int L1, int L2>
__device__ __forceinline__ void axis_table_compact(double za, double zb, double xab, double *E) {
    constexpr int NT = L1 + L2 + 1;
    double tmp[(L1 + 1) * (L2 + 1) * NT];
    axis_table<L1, L2>(za, zb, xab, tmp);
#pragma unroll
    for (int i = 0; i <= L1; ++i)
#pragma unroll
        for (int j = 0; j <= L2; ++j)
#pragma unroll
            for (int t = 0; t <= i + j; ++t) E[e1_rowoff(L2, i, j) + t] = tmp[(i * (L2 + 1) + j) * NT + t];
}

// Table record of one primitive pair: rec[0] = p, rec[1..3] = P, rec[4] = c_a c_b, rec[5] = -c_a c_b,
// rec[6] = 0, rec[7] = 1/p, rec[8 + ax*E1 + ..] = the compact 1-D tables (the slots prod_word addresses).
template <int L1, int L2>
__device__ __forceinline__ void table_task(const PairView &pv, long long i1, long long i2, int k1, int k2, int ax, double *rec) {
    constexpr int E1 = e1_count(L1, L2);
    const int K1 = pv.a.K, K2 = pv.b.K;
    const double za = __ldg(pv.a.exps + i1 * K1 + k1), A = __ldg(pv.a.center + 3 * i1 + ax);
    double zb = 0.0, B = A;
    if (!pv.single) { zb = __ldg(pv.b.exps + i2 * K2 + k2); B = __ldg(pv.b.center + 3 * i2 + ax); }
    axis_table_compact<L1, L2>(za, zb, A - B, rec + 8 + ax * E1);
    const double p = za + zb;
    rec[1 + ax] = (za * A + zb * B) / p;
    if (ax == 0) {
        rec[0] = p;
        const double c = __ldg(pv.a.coefs + i1 * K1 + k1) * (pv.single ? 1.0 : __ldg(pv.b.coefs + i2 * K2 + k2));
        rec[4] = c; rec[5] = -c; rec[6] = 0.0; rec[7] = 1.0 / p;
    }
}

// Eq. 24 along one direction.  a[0][m] = [..0..]^(m), m = 0..n, on entry; after step t the row
// a[(t+1)&1][m] holds [..t+1..]^(m), m = 0..n-t-1.  emit(t, row) is called for t = 0..n.
template <int N, class Emit>
__device__ __forceinline__ void line_recursion(double X, double (&a)[2][N + 1], int n, Emit &&emit) {
    emit(std::integral_constant<int, 0>{}, a[0]);
    static_for<N>([&](auto tc) {
        constexpr int t = decltype(tc)::value;
        if (t < n) {
            double(&cur)[N + 1] = a[t & 1];
            double(&nxt)[N + 1] = a[(t + 1) & 1];
#pragma unroll
            for (int m = 0; m < N - t; ++m) {
                double v = X * cur[m + 1];
                if (t > 0) v = fma((double)t, nxt[m + 1], v);
                nxt[m] = v;
            }
            emit(std::integral_constant<int, t + 1>{}, nxt);
        }
    });
}

template <int LA, int LB, int LC, int LD, bool PURE, int PB, int NCH>
struct F2Impl {
    using C = F2Cfg<LA, LB, LC, LD, PURE, PB, NCH>;
    static constexpr int L = C::L;

    // ---- producer stages -------------------------------------------------------------------
    // stage 1a: Boys function, [0]^(m) and the z-line for one tensor
    static __device__ __forceinline__ void z_task(const double *bt, const double *kt, double *gs, double *cb,
                                                  const double *boys_tab) {
        // bt, kt: bra and ket primitive-pair headers in the L2 scratch
        const double p = __ldcg(bt), q = __ldcg(kt), ipq = __ldcg(bt + 7) * __ldcg(kt + 7);
        const double X = __ldcg(bt + 1) - __ldcg(kt + 1), Y = __ldcg(bt + 2) - __ldcg(kt + 2), Z = __ldcg(bt + 3) - __ldcg(kt + 3);
        const double rs = rsqrt(p + q);                                    // no FP64 division on this path:
        const double rho = p * q * rs * rs;                                // rho = pq/(p+q)            (Eq. 23)
        const double T = rho * (X * X + Y * Y + Z * Z);
        // Boys function, every order from the Taylor table on its own (boys.cuh, scheme 1): the L+8 table
        // values are loaded once; the L+1 Horner chains are independent, so the chain is 8 FMAs deep.
        double F[L + 1];
        if (T < MD_BOYS_TASY) {
            const int i = __double2int_rn(T * MD_BOYS_ISTEP);
            const double mh = i * MD_BOYS_STEP - T;
            const double *row = boys_tab + i * MD_BOYS_MTAB;
            double r[L + 8];
#pragma unroll
            for (int k = 0; k < L + 8; ++k) r[k] = __ldg(row + k);
#pragma unroll
            for (int m = 0; m <= L; ++m) {
                double s = r[m + 7] * (1.0 / 5040.0);
                s = fma(s, mh, r[m + 6] * (1.0 / 720.0));
                s = fma(s, mh, r[m + 5] * (1.0 / 120.0));
                s = fma(s, mh, r[m + 4] * (1.0 / 24.0));
                s = fma(s, mh, r[m + 3] * (1.0 / 6.0));
                s = fma(s, mh, r[m + 2] * 0.5);
                s = fma(s, mh, r[m + 1]);
                F[m] = fma(s, mh, r[m]);
            }
        } else {
            const double it = 1.0 / T, h = 0.5 * it;
            double f = 0.88622692545275801365 * sqrt(it);
#pragma unroll
            for (int m = 0; m <= L; ++m) { F[m] = f; f *= (2 * m + 1) * h; }
        }
        double a[2][L + 1];
        double f = 34.98683665524972497 * ipq * rs;                       // 2 pi^{5/2}/(pq sqrt(p+q))   (Eq. 21)
        const double m2r = -2.0 * rho;
#pragma unroll
        for (int m = 0; m <= L; ++m) { a[0][m] = F[m] * f; f *= m2r; a[1][m] = 0.0; }
        gs[C::O_PQ] = X; gs[C::O_PQ + 1] = Y; gs[C::O_PQ + 2] = Z;
        double *zo = cb + C::O_R;
        line_recursion<L>(Z, a, L, [&](auto vc, double(&row)[L + 1]) {
            constexpr int v = decltype(vc)::value;
            constexpr int off = v * (L + 1) - v * (v - 1) / 2;
#pragma unroll
            for (int m = 0; m <= L - v; ++m) zo[off + m] = row[m];
        });
    }
    // stage y: thread owns v; [0uv]^(m) for u = 0..L-v, written as columns (u,v) of L-u-v+1 entries
    static __device__ __forceinline__ void y_task(int v, double *gs, const double *cb) {
        const int n = L - v;
        const double *zo = cb + C::O_R + v * (L + 1) - v * (v - 1) / 2;
        double a[2][L + 1];
#pragma unroll
        for (int m = 0; m <= L; ++m) { a[0][m] = m <= n ? zo[m] : 0.0; a[1][m] = 0.0; }
        double *col = gs + C::O_B + (nherm(L) - nherm(n));                 // block of this v
        line_recursion<L>(gs[C::O_PQ + 1], a, n, [&](auto uc, double(&row)[L + 1]) {
            constexpr int u = decltype(uc)::value;
#pragma unroll
            for (int m = 0; m <= L - u; ++m)
                if (m <= n - u) col[m] = row[m];
            col += n - u + 1;
        });
    }
    // stage x: thread owns the line (u,v); emits [tuv]^(0) into the brick layout (fused2_tables.cuh)
    static __device__ __forceinline__ void x_task(int u, int v, const double *gs, double *cb) {
        const int nv = L - v, n = nv - u;
        const double *col = gs + C::O_B + (nherm(L) - nherm(nv)) + u * (nv + 1) - u * (u - 1) / 2;
        double a[2][L + 1];
#pragma unroll
        for (int m = 0; m <= L; ++m) { a[0][m] = m <= n ? col[m] : 0.0; a[1][m] = 0.0; }
        double *R = cb + C::O_R + C::BR.B * u + v;
        line_recursion<L>(gs[C::O_PQ], a, n, [&](auto tc, double(&row)[L + 1]) {
            constexpr int t = decltype(tc)::value;
            R[C::BR.A * t] = row[0];
        });
    }
    // products of one Cartesian component pair, written at the positions POS gives
    template <int L1, int L2, bool SIGN, class POS>
    static __device__ __forceinline__ void prod_task(const double *tab, int comp, double *dst, POS &&pos) {
        constexpr int NC2 = ncart(L2), E1 = e1_count(L1, L2);
        const int c = comp / NC2, d = comp - c * NC2;
        const int ea = d_cart<L1>.e[c], eb = d_cart<L2>.e[d];
        const int ax = ea & 0xff, ay = ea >> 8 & 0xff, az = ea >> 16, bx = eb & 0xff, by = eb >> 8 & 0xff, bz = eb >> 16;
        const short *ro = d_e1row<L1, L2>.off;
        const double *Ex = tab + 8 + ro[ax * (L2 + 1) + bx];
        const double *Ey = tab + 8 + E1 + ro[ay * (L2 + 1) + by];
        const double *Ez = tab + 8 + 2 * E1 + ro[az * (L2 + 1) + bz];
        const double coef = tab[4];
        int i = 0;
        for (int t = 0; t <= ax + bx; ++t) {
            const double et = coef * Ex[t];
            for (int u = 0; u <= ay + by; ++u) {
                const double eu = et * Ey[u];
                for (int v = 0; v <= az + bz; ++v, ++i) {
                    double val = eu * Ez[v];
                    if (SIGN && ((t + u + v) & 1)) val = -val;
                    dst[pos(comp, i)] = val;
                }
            }
        }
    }
};

}  // namespace mdb
