// lowl.cuh -- one THREAD per quartet for the store-bound classes with every l <= 1 ((ss|ss) .. (pp|pp), (ss|s) .. (pp|p)).
//
// PAPER.md:204-210 (V0: "all but the final results reside in registers"), 143-146, 188 (128-byte transactions): these
// classes do a few hundred flops per quartet and are bound by moving 8 N_ab N_cd bytes out and four shells in.  Here
//   * a thread evaluates S1-S5 for its quartet entirely in registers with compile-time l (every loop below unrolls to
//     straight-line code; coefficients that vanish by Eq. 14 are never formed);
//   * the N_ab N_cd results of the 32 quartets of a warp go to a padded shared-memory tile [component][33] and leave as
//     ONE contiguous run of 32 N_ab N_cd doubles, so every store instruction writes full 128-byte lines;
//   * inputs are read straight from the caller's structure-of-arrays shell batches.
// Quartet-major layout only (list or product mode); the paper layout stays with the fused kernels.
#pragma once
#include "boys.cuh"
#include "common.cuh"

namespace mdb {

struct LowlArgs {
    PairView bra, ket;
    const int32_t *qidx;
    long long nq, nket;
    double *out;
    int pure;
    const double *boys_tab;
};

#define MD_LOWL_THREADS 128

// index of (t,u,v) in the degree-sorted Hermite list (common.cuh), usable in constant expressions
__host__ __device__ constexpr int lw_hidx(int t, int u, int v) { return herm_index(t, u, v); }

// [tuv]^(0) for t+u+v <= L from F_m(T) (Eqs. 21, 24), level by level in registers: lvl(m) holds [r~]^(m) for
// |r~| <= L-m.  pref = 2 pi^{5/2}/(p q sqrt(p+q)) times the four coefficients; m2r = -2 rho.
template <int L>
__device__ __forceinline__ void lw_hermite_R(const double (&F)[L + 1], double pref, double m2r, const double (&PQ)[3],
                                             double (&R)[nherm(L)]) {
    double cur[nherm(L)], nxt[nherm(L)];
    double g[L + 1];
    double f = pref;
#pragma unroll
    for (int m = 0; m <= L; ++m) { g[m] = f * F[m]; f *= m2r; }
    cur[0] = g[L];
#pragma unroll
    for (int m = L - 1; m >= 0; --m) {
        nxt[0] = g[m];
#pragma unroll
        for (int n = 1; n <= L - m; ++n)
#pragma unroll
            for (int t = n; t >= 0; --t)
#pragma unroll
                for (int u = n - t; u >= 0; --u) {
                    const int v = n - t - u;
                    double val;
                    if (t > 0) {
                        val = PQ[0] * cur[lw_hidx(t - 1, u, v)];
                        if (t > 1) val = fma((double)(t - 1), cur[lw_hidx(t - 2, u, v)], val);
                    } else if (u > 0) {
                        val = PQ[1] * cur[lw_hidx(t, u - 1, v)];
                        if (u > 1) val = fma((double)(u - 1), cur[lw_hidx(t, u - 2, v)], val);
                    } else {
                        val = PQ[2] * cur[lw_hidx(t, u, v - 1)];
                        if (v > 1) val = fma((double)(v - 1), cur[lw_hidx(t, u, v - 2)], val);
                    }
                    nxt[lw_hidx(t, u, v)] = val;
                }
#pragma unroll
        for (int e = 0; e < nherm(L - m); ++e) cur[e] = nxt[e];
    }
#pragma unroll
    for (int e = 0; e < nherm(L); ++e) R[e] = cur[e];
}

// 1-D Hermite coefficients of one axis for i, j <= 1 (Eqs. 9, 10, 13 without the exponential, which goes into the
// prefactor): E[i][j][t], t <= i+j.  xpa = (P-A), xpb = (P-B), h = 1/(2p).
struct LwAxis { double e[2][2][3]; };
__device__ __forceinline__ LwAxis lw_axis(double xpa, double xpb, double h) {
    LwAxis a;
    a.e[0][0][0] = 1.0; a.e[0][0][1] = 0.0; a.e[0][0][2] = 0.0;
    a.e[1][0][0] = xpa; a.e[1][0][1] = h;   a.e[1][0][2] = 0.0;
    a.e[0][1][0] = xpb; a.e[0][1][1] = h;   a.e[0][1][2] = 0.0;
    a.e[1][1][0] = fma(xpa, xpb, h); a.e[1][1][1] = (xpa + xpb) * h; a.e[1][1][2] = h * h;
    return a;
}

// Cartesian exponents of component k of shell l <= 1, and its position in the output (solid order of p is y, z, x).
__host__ __device__ constexpr int lw_exp(int l, int k, int axis) { return l == 0 ? 0 : (k == axis ? 1 : 0); }
__host__ __device__ constexpr int lw_pos(int l, int k, bool pure) { return (l == 1 && pure) ? (k + 2) % 3 : k; }

// Occupancy: the kernel is bound by the latency of its input loads, so the small classes trade registers for resident warps.
__host__ __device__ constexpr int lw_min_blocks(int nout) { return nout <= 3 ? 8 : nout <= 9 ? 6 : nout <= 27 ? 4 : 2; }

template <int LA, int LB, int LC, int LD, bool SINGLE>
__global__ void __launch_bounds__(MD_LOWL_THREADS, lw_min_blocks((2 * LA + 1) * (2 * LB + 1) * (2 * LC + 1) * (2 * LD + 1)))
lowl_kernel(LowlArgs g) {
    constexpr int NA = 2 * LA + 1, NB = 2 * LB + 1, NC = 2 * LC + 1, ND = 2 * LD + 1;   // Cartesian = solid count for l <= 1
    constexpr int NOUT = NA * NB * NC * ND, Lb = LA + LB, Lk = LC + LD, L = Lb + Lk;
    extern __shared__ double sm[];
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    double *tile = sm + (size_t)warp * NOUT * 33;                     // [component][33]
    const int Ka = g.bra.a.K, Kb = g.bra.b.K, Kc = g.ket.a.K, Kd = SINGLE ? 1 : g.ket.b.K;
    const bool pure = g.pure != 0;
    const long long nwarps_total = (long long)gridDim.x * (MD_LOWL_THREADS / 32);
    for (long long q0 = ((long long)blockIdx.x * (MD_LOWL_THREADS / 32) + warp) * 32; q0 < g.nq; q0 += nwarps_total * 32) {
        const long long q = q0 + lane;
        const bool live = q < g.nq;
        const long long qq = live ? q : g.nq - 1;
        long long bi, ki;
        if (g.qidx) { bi = g.qidx[2 * qq]; ki = g.qidx[2 * qq + 1]; }
        else { bi = qq / g.nket; ki = qq % g.nket; }
        long long ia = bi, ib = bi, ic = ki, id = ki;
        if (g.bra.idx) { ia = g.bra.idx[2 * bi]; ib = g.bra.idx[2 * bi + 1]; }
        if (g.ket.idx) { ic = g.ket.idx[2 * ki]; id = g.ket.idx[2 * ki + 1]; }
        double A[3], B[3], C[3], D[3];
#pragma unroll
        for (int x = 0; x < 3; ++x) {
            A[x] = g.bra.a.center[3 * ia + x]; B[x] = g.bra.b.center[3 * ib + x];
            C[x] = g.ket.a.center[3 * ic + x]; D[x] = SINGLE ? C[x] : g.ket.b.center[3 * id + x];
        }
        const double ab2 = (A[0] - B[0]) * (A[0] - B[0]) + (A[1] - B[1]) * (A[1] - B[1]) + (A[2] - B[2]) * (A[2] - B[2]);
        const double cd2 = (C[0] - D[0]) * (C[0] - D[0]) + (C[1] - D[1]) * (C[1] - D[1]) + (C[2] - D[2]) * (C[2] - D[2]);
        const bool one = Ka * Kb * Kc * Kd == 1;                      // uncontracted: results go straight to the tile
        if (!one) {
#pragma unroll
            for (int i = 0; i < NOUT; ++i) tile[i * 33 + lane] = 0.0;
        }
        for (int kab = 0; kab < Ka * Kb; ++kab) {
            const int ka = kab / Kb, kb = kab - ka * Kb;
            const double za = g.bra.a.exps[ia * Ka + ka], zb = g.bra.b.exps[ib * Kb + kb];
            const double p = za + zb, ip = 1.0 / p, hp = 0.5 * ip;
            const double cab = g.bra.a.coefs[ia * Ka + ka] * g.bra.b.coefs[ib * Kb + kb] * exp(-za * zb * ip * ab2);   // Eq. 13
            double P[3];
            LwAxis eb[3];
#pragma unroll
            for (int x = 0; x < 3; ++x) {
                P[x] = (za * A[x] + zb * B[x]) * ip;
                eb[x] = lw_axis(P[x] - A[x], P[x] - B[x], hp);
            }
            for (int kcd = 0; kcd < Kc * Kd; ++kcd) {
                const int kc = kcd / Kd, kd = kcd - kc * Kd;
                const double zc = g.ket.a.exps[ic * Kc + kc], zd = SINGLE ? 0.0 : g.ket.b.exps[id * Kd + kd];
                const double qe = zc + zd, iq = 1.0 / qe, hq = 0.5 * iq;
                const double ccd = g.ket.a.coefs[ic * Kc + kc] * (SINGLE ? 1.0 : g.ket.b.coefs[id * Kd + kd] * exp(-zc * zd * iq * cd2));
                double PQ[3];
                LwAxis ek[3];
#pragma unroll
                for (int x = 0; x < 3; ++x) {
                    const double Qx = (zc * C[x] + zd * D[x]) * iq;
                    ek[x] = lw_axis(Qx - C[x], Qx - D[x], hq);
                    PQ[x] = P[x] - Qx;
                }
                const double rho = p * qe / (p + qe);
                const double T = rho * (PQ[0] * PQ[0] + PQ[1] * PQ[1] + PQ[2] * PQ[2]);
                double F[L + 1], R[nherm(L)];
                boys_eval_t<L>(T, g.boys_tab, F);
                lw_hermite_R<L>(F, 34.98683665524972497 * cab * ccd / (p * qe * sqrt(p + qe)), -2.0 * rho, PQ, R);   // Eq. 21
                // Eqs. 25-26 with the sparse Cartesian E (products of three axis entries); (-1)^{|q~|} of Eq. 19
#pragma unroll
                for (int c = 0; c < NC; ++c)
#pragma unroll
                    for (int d = 0; d < ND; ++d) {
                        double gp[nherm(Lb)];                         // [p~|cd]
#pragma unroll
                        for (int e = 0; e < nherm(Lb); ++e) gp[e] = 0.0;
#pragma unroll
                        for (int t2 = 0; t2 <= lw_exp(LC, c, 0) + lw_exp(LD, d, 0); ++t2)
#pragma unroll
                            for (int u2 = 0; u2 <= lw_exp(LC, c, 1) + lw_exp(LD, d, 1); ++u2)
#pragma unroll
                                for (int v2 = 0; v2 <= lw_exp(LC, c, 2) + lw_exp(LD, d, 2); ++v2) {
                                    double ecd = ek[0].e[lw_exp(LC, c, 0)][lw_exp(LD, d, 0)][t2] *
                                                 ek[1].e[lw_exp(LC, c, 1)][lw_exp(LD, d, 1)][u2] *
                                                 ek[2].e[lw_exp(LC, c, 2)][lw_exp(LD, d, 2)][v2];
                                    if ((t2 + u2 + v2) & 1) ecd = -ecd;
#pragma unroll
                                    for (int n = 0; n <= Lb; ++n)
#pragma unroll
                                        for (int t = n; t >= 0; --t)
#pragma unroll
                                            for (int u = n - t; u >= 0; --u)
                                                gp[lw_hidx(t, u, n - t - u)] = fma(ecd, R[lw_hidx(t + t2, u + u2, n - t - u + v2)],
                                                                                   gp[lw_hidx(t, u, n - t - u)]);
                                }
#pragma unroll
                        for (int a = 0; a < NA; ++a)
#pragma unroll
                            for (int b = 0; b < NB; ++b) {
                                double s = 0.0;
#pragma unroll
                                for (int t = 0; t <= lw_exp(LA, a, 0) + lw_exp(LB, b, 0); ++t)
#pragma unroll
                                    for (int u = 0; u <= lw_exp(LA, a, 1) + lw_exp(LB, b, 1); ++u)
#pragma unroll
                                        for (int v = 0; v <= lw_exp(LA, a, 2) + lw_exp(LB, b, 2); ++v)
                                            s = fma(eb[0].e[lw_exp(LA, a, 0)][lw_exp(LB, b, 0)][t] *
                                                    eb[1].e[lw_exp(LA, a, 1)][lw_exp(LB, b, 1)][u] *
                                                    eb[2].e[lw_exp(LA, a, 2)][lw_exp(LB, b, 2)][v], gp[lw_hidx(t, u, v)], s);
                                // component positions: Cartesian order x,y,z; solid order of a p shell is y,z,x (m = -1,0,1)
                                const int pc = ((lw_pos(LA, a, true) * NB + lw_pos(LB, b, true)) * NC + lw_pos(LC, c, true)) * ND + lw_pos(LD, d, true);
                                const int cc = ((a * NB + b) * NC + c) * ND + d;
                                double *o = tile + (pure ? pc : cc) * 33 + lane;
                                if (one) *o = s; else *o += s;
                            }
                    }
            }
        }
        __syncwarp();
        // the warp's 32 quartets are one contiguous run of the quartet-major output
        const long long nvalid = min(32LL, g.nq - q0) * NOUT;
        double *o = g.out + q0 * NOUT;
        for (int i = lane; i < nvalid; i += 32) {
            const int ql = i / NOUT, comp = i - ql * NOUT;
            o[i] = tile[comp * 33 + ql];
        }
        __syncwarp();
    }
}

}  // namespace mdb
