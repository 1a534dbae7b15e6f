// pair.cuh -- step S1 of the hot path for the runtime-l kernel chain: primitive-pair setup.
//
// For every shell pair (a,b) of a pair batch and every primitive pair (ka,kb) this kernel
// writes one record of `stride` doubles ("{G, H[ab,p]}[ij,K_b]" stored
// contiguously per pair and primitive):
//   rec[0]    = p = zeta_a + zeta_b
//   rec[1..3] = P = (zeta_a A + zeta_b B)/p
//   rec[4 + p~*N_ab + ab] = H[p~][ab]
// with H the Hermite->AO matrix of PAPER.md Eqs. 7 and 17,
//   Cartesian: H[p~][ab]   = c_a c_b E^{t}_{ax bx} E^{u}_{ay by} E^{v}_{az bz}
//   solid    : H[p~][mamb] = sum_{a,b} C^{la}_{ma,a} C^{lb}_{mb,b} H[p~][ab]   (Eq. 17)
// stored p~-major so that both Hermite->AO contractions read one contiguous row per Hermite
// index.  For the ket batch the factor (-1)^{|q~|} of Eq. 19 is folded in (ket_sign = 1).
// A one-centre batch (3-center X, Eqs. 6, 8, 11, 12) is the same recursion with
// zeta_b = 0, c_b = 1, B = A (Eq. 8 is Eq. 9 at P = A; reading G2).
#pragma once
#include "common.cuh"

namespace mdb {

// The 1-D tables E[(i*(lb+1)+j)*nt + t], nt = la+lb+1 (Eqs. 9, 10, 13, 14) come from hl_e_axis_warp (common.cuh), one warp per axis.

struct PairSetupArgs {
    PairView pv;
    int pure;
    int ket_sign;            // fold (-1)^{|q~|} (Eq. 19) into H
    int pchunk;              // Hermite rows per shared-memory chunk of the solid transform
    long long stride;        // doubles per (pair, primitive) record
    double *rec;             // [npairs][Ka*Kb][stride]
    // chunked list mode (md_b200.cu::run_generic): record r belongs to the bra (side 0) or ket (side 1) pair of quartet q0 + r
    const int32_t *by_quartet = nullptr;
    long long q0 = 0;
    int side = 0;
};

// One CTA per (pair, primitive pair).  Shared memory: 3 axis tables + the stage-A buffer.
// LM = max(la, lb) sizes the register rows of the solid transform (one instantiation per LM).
template <int LM>
__global__ void __launch_bounds__(128) pair_setup_kernel(PairSetupArgs g) {
    extern __shared__ double sm[];
    const PairView &pv = g.pv;
    const int la = pv.a.l, lb = pv.single ? 0 : pv.b.l;
    const int Ka = pv.a.K, Kb = pv.single ? 1 : pv.b.K;
    const int Lb = la + lb, nt = Lb + 1, nh = nherm(Lb);
    const int esz = (la + 1) * (lb + 1) * nt;
    double *E = sm;                     // [3][esz]
    double *T1 = sm + 3 * esz;          // [pchunk][nca][nb_out]
    __shared__ double hdr[5];           // p, P, coefficient
    // Lane-varying reads of __constant__ tables serialise (one transaction per distinct address), which made this
    // kernel 30x slower than its instruction count; the tables it needs are staged in shared memory instead.
    __shared__ uint32_t s_herm[455];                  // N~(12): Hermite triples up to order la+lb <= 12
    __shared__ double s_Ca[13 * 28], s_Cb[13 * 28];   // Cartesian -> solid matrices of the two shells
    for (int i = threadIdx.x; i < nh; i += blockDim.x) s_herm[i] = c_herm[i];
    for (int i = threadIdx.x; i < nsolid(la) * ncart(la); i += blockDim.x) s_Ca[i] = c_solid[solid_off(la) + i];
    for (int i = threadIdx.x; i < nsolid(lb) * ncart(lb); i += blockDim.x) s_Cb[i] = c_solid[solid_off(lb) + i];

    const long long rid = blockIdx.x;   // pair * Ka*Kb + prim
    long long ipair = rid / (Ka * Kb);
    if (g.by_quartet) ipair = g.by_quartet[2 * (g.q0 + ipair) + g.side];
    const int kp = (int)(rid % (Ka * Kb)), ka = kp / Kb, kb = kp % Kb;
    long long ia = ipair, ib = ipair;
    if (pv.idx) { ia = pv.idx[2 * ipair]; ib = pv.idx[2 * ipair + 1]; }

    if (threadIdx.x < 96) {             // one WARP per Cartesian axis (lane = t, neighbours by shuffle): a single thread per axis
        const int ax = threadIdx.x >> 5, lane = threadIdx.x & 31;   // took as long as the whole H build behind it ((ff|: 350 dependent DFMAs)
        double za = pv.a.exps[ia * Ka + ka], A = pv.a.center[3 * ia + ax];
        double zb = 0.0, B = A;
        if (!pv.single) { zb = pv.b.exps[ib * Kb + kb]; B = pv.b.center[3 * ib + ax]; }
        hl_e_axis_warp(la, lb, za, zb, A - B, E + ax * esz, lane);
        if (lane == 0) {
            double p = za + zb;
            hdr[1 + ax] = (za * A + zb * B) / p;
            if (ax == 0) {
                hdr[0] = p;
                hdr[4] = pv.a.coefs[ia * Ka + ka] * (pv.single ? 1.0 : pv.b.coefs[ib * Kb + kb]);
            }
        }
    }
    __syncthreads();
    double *rec = g.rec + rid * g.stride;
    if (threadIdx.x < 4) rec[threadIdx.x] = hdr[threadIdx.x];
    const double coef = hdr[4];
    const int nca = ncart(la), ncb = ncart(lb);
    const uint32_t *ca = s_herm + nherm(la - 1), *cb = s_herm + nherm(lb - 1);   // component exponents
    const double *Ex = E, *Ey = E + esz, *Ez = E + 2 * esz;
    double *H = rec + 4;

    if (!g.pure) {
        const int nab = nca * ncb;
        for (int e = threadIdx.x; e < nh * nab; e += blockDim.x) {
            int ih = e / nab, ab = e % nab, a = ab / ncb, b = ab % ncb;
            int t, u, v, ax, ay, az, bx, by, bz;
            unpack_tuv(s_herm[ih], t, u, v);
            unpack_tuv(ca[a], ax, ay, az);
            unpack_tuv(cb[b], bx, by, bz);
            double val = coef * Ex[(ax * (lb + 1) + bx) * nt + t] * Ey[(ay * (lb + 1) + by) * nt + u] *
                         Ez[(az * (lb + 1) + bz) * nt + v];
            if (g.ket_sign && ((t + u + v) & 1)) val = -val;
            H[e] = val;
        }
        return;
    }
    if (pv.single) {
        // One-centre solid harmonics (Hobson): S_lm(d/dA) e^{-z r_A^2} = (2z)^l S_lm(r_A) e^{-z r_A^2}, so
        // only the Hermites of order exactly l appear, with coefficient C^l_{m,q~}/(2z)^l.  Writing the
        // zeros exactly (instead of leaving Eq. 17's cancellation to rounding) keeps the result accurate
        // relative to the small solid block (finding F1).
        const int nsa = nsolid(la), nlow = nherm(la - 1);
        const double *Ca = s_Ca;
        double f = coef;
        for (int i = 0; i < la; ++i) f *= 0.5 / hdr[0];
        if (g.ket_sign && (la & 1)) f = -f;
        for (int e = threadIdx.x; e < nh * nsa; e += blockDim.x) {
            int ih = e / nsa, m = e % nsa;
            H[e] = ih < nlow ? 0.0 : f * Ca[m * nca + (ih - nlow)];
        }
        return;
    }
    // Solid harmonics, Eq. 17, one index at a time, pchunk Hermite rows per pass, register-blocked:
    //   stage A  thread (p~, a): the Cartesian row E^{ab}_{p~}, b = 0..ncb-1, in registers (Eq. 7, zeros by Eq. 14),
    //            then T1[p~][a][mb] = sum_b C^{lb}[mb][b] E^{ab}_{p~}
    //   stage B  thread (p~, mb): the column T1[p~][.][mb] in registers,
    //            then H[p~][ma][mb] = coef * sum_a C^{la}[ma][a] T1[p~][a][mb]
    constexpr int NCMAX = (LM + 1) * (LM + 2) / 2;
    const int nsa = nsolid(la), nsb = nsolid(lb);
    const double *Ca = s_Ca, *Cb = s_Cb;
    for (int h0 = 0; h0 < nh; h0 += g.pchunk) {
        const int hc = min(g.pchunk, nh - h0);
        for (int e = threadIdx.x; e < hc * nca; e += blockDim.x) {
            const int ih = e / nca, a = e - ih * nca;
            int t, u, v, ax, ay, az;
            unpack_tuv(s_herm[h0 + ih], t, u, v);
            unpack_tuv(ca[a], ax, ay, az);
            const double *ex = Ex + ax * (lb + 1) * nt + t, *ey = Ey + ay * (lb + 1) * nt + u, *ez = Ez + az * (lb + 1) * nt + v;
            double row[NCMAX];
#pragma unroll
            for (int b = 0; b < NCMAX; ++b) {
                double x = 0.0;
                if (b < ncb) {
                    int bx, by, bz;
                    unpack_tuv(cb[b], bx, by, bz);
                    if (t <= ax + bx && u <= ay + by && v <= az + bz) x = ex[bx * nt] * ey[by * nt] * ez[bz * nt];
                }
                row[b] = x;
            }
            double *dst = T1 + (size_t)e * nsb;
            for (int mb = 0; mb < nsb; ++mb) {
                const double *c = Cb + mb * ncb;
                double s0 = 0.0;
#pragma unroll
                for (int b = 0; b < NCMAX; ++b)
                    if (b < ncb) s0 = fma(c[b], row[b], s0);
                dst[mb] = s0;
            }
        }
        __syncthreads();
        for (int e = threadIdx.x; e < hc * nsb; e += blockDim.x) {
            const int ih = e / nsb, mb = e - ih * nsb;
            const double *t1 = T1 + (size_t)ih * nca * nsb + mb;
            double col[NCMAX];
#pragma unroll
            for (int a = 0; a < NCMAX; ++a) col[a] = a < nca ? t1[a * nsb] : 0.0;
            const bool neg = g.ket_sign && (s_herm[h0 + ih] >> 24 & 1);
            double *dst = H + (long long)(h0 + ih) * nsa * nsb + mb;
            for (int ma = 0; ma < nsa; ++ma) {
                const double *c = Ca + ma * nca;
                double s0 = 0.0;
#pragma unroll
                for (int a = 0; a < NCMAX; ++a)
                    if (a < nca) s0 = fma(c[a], col[a], s0);
                s0 *= coef;
                dst[(long long)ma * nsb] = neg ? -s0 : s0;
            }
        }
        __syncthreads();
    }
}

}  // namespace mdb
