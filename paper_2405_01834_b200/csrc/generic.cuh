// generic.cuh -- runtime-l quartet kernel: steps S2-S5 for every class with l <= 6, any K,
// 3- and 4-center, Cartesian or solid output.  One CTA per quartet (grid-stride).
//
// Per primitive quartet (kb over bra primitives, kk over ket primitives):
//   S2  rho = pq/(p+q), T = rho |P-Q|^2, F_m(T), m = 0..L              (Eqs. 22-23)
//       [0]^(m) = (-2 rho)^m 2 pi^{5/2}/(pq sqrt(p+q)) F_m(T)          (Eq. 21)
//   S3  [r+1_i]^(m) = r_i [r-1_i]^(m+1) + (P_i-Q_i) [r]^(m+1)          (Eq. 24; readings G5, G6)
//       level by level in place in shared memory, [r]^(0) for |r| <= L
//   S4  [p~|cd] = sum_q~ [p~+q~]^(0) Hk[q~][cd]       (Eqs. 19, 25; the sign (-1)^{|q~|} is in Hk)
//       [ab|cd] += sum_p~ Hb[p~][ab] [p~|cd]          (Eq. 26)
//   S5  the solid-harmonic matrices are already folded into Hb and Hk by pair_setup_kernel
//       (Eq. 17), so S4 lands directly in the output components; store.
// [r]^(0) is kept as a dense cube R[(t*S+u)*S+v], S = L+1, so that the Hankel structure of
// Eq. 19 is an index ADDITION: cube(p~+q~) = cube(p~) + cube(q~).
// The half-transformed block [p~|cd] is tiled over cd (ct columns per pass) to fit shared
// memory; with K_ket > 1 each primitive quartet is pushed through both contractions and
// accumulated in the output (plain read-modify-write: the CTA owns its quartet).
#pragma once
#include "boys.cuh"
#include "common.cuh"

namespace mdb {

struct GenericArgs {
    const double *rec_bra, *rec_ket;     // pair_setup_kernel records
    long long stride_bra, stride_ket;
    int Kbra, Kket;                      // primitive pairs per shell pair (Ka*Kb, Kc*Kd)
    int Lb, Lk, nab, ncd;                // N_ab, N_cd in the output components
    int ct;                              // cd-tile width
    const int32_t *qidx;                 // [nq][2] or nullptr (product, ket fastest)
    long long nq, nket;
    double *out;
    long long s_q, s_bi, s_ki, s_ab, s_cd;   // out[q*s_q + bi*s_bi + ki*s_ki + ab*s_ab + cd*s_cd]
    const double *boys_tab;
};

#define MD_GEN_THREADS 256
#define MD_GEN_RPT 12                    // ceil(N~(24)/256): cube entries per thread per level

__global__ void __launch_bounds__(MD_GEN_THREADS) eri_generic_kernel(GenericArgs g) {
    extern __shared__ double sm[];
    const int L = g.Lb + g.Lk, S = L + 1;
    const int nhb = nherm(g.Lb), nhk = nherm(g.Lk);
    double *R = sm;                               // [S^3]
    double *half = R + S * S * S;                 // [nhb][ct]
    double *G0 = half + (size_t)nhb * g.ct;       // [L+1]  [0]^(m)
    int *cube_b = (int *)(G0 + S + (S & 1));      // [nhb] cube index of p~
    int *cube_k = cube_b + nhb;                   // [nhk] cube index of q~
    __shared__ double pq[3];
    const int tid = threadIdx.x;

    for (int e = tid; e < nhb + nhk; e += MD_GEN_THREADS) {
        int t, u, v;
        unpack_tuv(c_herm[e < nhb ? e : e - nhb], t, u, v);
        cube_b[e] = (t * S + u) * S + v;          // cube_k follows cube_b contiguously
    }

    for (long long q = blockIdx.x; q < g.nq; q += gridDim.x) {
        long long bi, ki;
        if (g.qidx) { bi = g.qidx[2 * q]; ki = g.qidx[2 * q + 1]; }
        else { bi = q / g.nket; ki = q % g.nket; }
        double *out = g.out + q * g.s_q + bi * g.s_bi + ki * g.s_ki;

        for (int kb = 0; kb < g.Kbra; ++kb)
        for (int kk = 0; kk < g.Kket; ++kk) {
            const double *rb = g.rec_bra + (bi * g.Kbra + kb) * g.stride_bra;
            const double *rk = g.rec_ket + (ki * g.Kket + kk) * g.stride_ket;
            __syncthreads();                      // previous primitive quartet is done with R, G0
            if (tid == 0) {
                double p = rb[0], qq = rk[0];
                double X = rb[1] - rk[1], Y = rb[2] - rk[2], Z = rb[3] - rk[3];
                double rho = p * qq / (p + qq);
                boys_eval(L, rho * (X * X + Y * Y + Z * Z), g.boys_tab, G0);
                double f = 34.98683665524972497 / (p * qq * sqrt(p + qq));   // 2 pi^{5/2}
                for (int m = 0; m <= L; ++m) { G0[m] *= f; f *= -2.0 * rho; }
                pq[0] = X; pq[1] = Y; pq[2] = Z;
                R[0] = G0[L];
            }
            __syncthreads();
            // S3: level m holds [r]^(m) for |r| <= L-m; computed from level m+1, in place.
            const double X = pq[0], Y = pq[1], Z = pq[2];
            for (int m = L - 1; m >= 0; --m) {
                const int ne = nherm(L - m);
                double tmp[MD_GEN_RPT];
#pragma unroll
                for (int k = 0; k < MD_GEN_RPT; ++k) {
                    int e = tid + k * MD_GEN_THREADS;
                    if (e < ne) {
                        int t, u, v;
                        unpack_tuv(c_herm[e], t, u, v);
                        int c = (t * S + u) * S + v;
                        double val;
                        if (t > 0) {
                            val = X * R[c - S * S];
                            if (t > 1) val += (t - 1) * R[c - 2 * S * S];
                        } else if (u > 0) {
                            val = Y * R[c - S];
                            if (u > 1) val += (u - 1) * R[c - 2 * S];
                        } else if (v > 0) {
                            val = Z * R[c - 1];
                            if (v > 1) val += (v - 1) * R[c - 2];
                        } else {
                            val = G0[m];
                        }
                        tmp[k] = val;
                    }
                }
                __syncthreads();
#pragma unroll
                for (int k = 0; k < MD_GEN_RPT; ++k) {
                    int e = tid + k * MD_GEN_THREADS;
                    if (e < ne) {
                        int t, u, v;
                        unpack_tuv(c_herm[e], t, u, v);
                        R[(t * S + u) * S + v] = tmp[k];
                    }
                }
                __syncthreads();
            }
            // S4, tiled over cd.
            const double *Hb = rb + 4, *Hk = rk + 4;
            const bool first = (kb == 0 && kk == 0);
            for (int cd0 = 0; cd0 < g.ncd; cd0 += g.ct) {
                const int ct = min(g.ct, g.ncd - cd0);
                // [p~|cd] = sum_q~ R[cube(p~)+cube(q~)] Hk[q~][cd]; 4 rows x 1 column per work item
                const int nrb = (nhb + 3) / 4;
                for (int it = tid; it < nrb * ct; it += MD_GEN_THREADS) {
                    const int r0 = (it / ct) * 4, c = it % ct;
                    int b0 = cube_b[r0], b1 = cube_b[min(r0 + 1, nhb - 1)], b2 = cube_b[min(r0 + 2, nhb - 1)],
                        b3 = cube_b[min(r0 + 3, nhb - 1)];
                    double a0 = 0, a1 = 0, a2 = 0, a3 = 0;
                    const double *hk = Hk + cd0 + c;
                    for (int iq = 0; iq < nhk; ++iq) {
                        double h = hk[(size_t)iq * g.ncd];
                        int cq = cube_k[iq];
                        a0 = fma(R[b0 + cq], h, a0);
                        a1 = fma(R[b1 + cq], h, a1);
                        a2 = fma(R[b2 + cq], h, a2);
                        a3 = fma(R[b3 + cq], h, a3);
                    }
                    half[(size_t)r0 * g.ct + c] = a0;
                    if (r0 + 1 < nhb) half[(size_t)(r0 + 1) * g.ct + c] = a1;
                    if (r0 + 2 < nhb) half[(size_t)(r0 + 2) * g.ct + c] = a2;
                    if (r0 + 3 < nhb) half[(size_t)(r0 + 3) * g.ct + c] = a3;
                }
                __syncthreads();
                // [ab|cd] += sum_p~ Hb[p~][ab] [p~|cd]; 2 rows x 1 column per work item
                const int nra = (g.nab + 1) / 2;
                for (int it = tid; it < nra * ct; it += MD_GEN_THREADS) {
                    const int ab0 = (it / ct) * 2, c = it % ct;
                    const int ab1 = min(ab0 + 1, g.nab - 1);
                    double a0 = 0, a1 = 0;
                    for (int ip = 0; ip < nhb; ++ip) {
                        double hv = half[(size_t)ip * g.ct + c];
                        a0 = fma(Hb[(size_t)ip * g.nab + ab0], hv, a0);
                        a1 = fma(Hb[(size_t)ip * g.nab + ab1], hv, a1);
                    }
                    double *o0 = out + ab0 * g.s_ab + (cd0 + c) * g.s_cd;
                    double *o1 = out + ab1 * g.s_ab + (cd0 + c) * g.s_cd;
                    if (first) { *o0 = a0; if (ab0 + 1 < g.nab) *o1 = a1; }
                    else { *o0 += a0; if (ab0 + 1 < g.nab) *o1 += a1; }
                }
                __syncthreads();
            }
        }
    }
}

}  // namespace mdb
