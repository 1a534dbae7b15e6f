// warp.cuh -- runtime-l quartet kernel for SMALL classes: one warp per quartet, no CTA barrier.
//
// The DMMA kernel gives a whole CTA to one quartet; for classes whose half-transformed block [p~|cd] has a few
// hundred entries (an s or p pair on one side, a fitting shell, (ss|X), (ab|ss) ...) that leaves most of the
// CTA idle and the quartet rate far below what the paper reports for the same shapes (profiles/r01_sweep_paper.md).
// Here each warp owns a quartet: the lanes evaluate F_m(T) for m = 0..L (one order per lane), build the
// Hermite Coulomb tensor level by level in the warp's own shared memory (Eqs. 21-24, __syncwarp only),
// and run the two Hermite->AO contractions (Eqs. 19, 25, 26) as DFMA loops over the dense H matrices of
// pair_setup_kernel, one output element per lane at a time.  L = la+lb+lc+ld <= 12.
#pragma once
#include "boys.cuh"
#include "common.cuh"
#include "mma.cuh"          // herm_index_packed

namespace mdb {

#define MD_WARP_THREADS 256
#define MD_WARP_LMAX 12
#define MD_WARP_HALF 640                 // largest [p~|cd] block (doubles) a warp keeps

struct WarpArgs {
    const double *rec_bra, *rec_ket;     // pair_setup_kernel records
    long long stride_bra, stride_ket;
    int Kbra, Kket;
    int Lb, Lk, nab, ncd;
    int kq0;                             // first ket Hermite row with a non-zero H (one-centre solid kets)
    const int32_t *qidx;
    long long nq, nket;
    double *out;
    long long s_q, s_bi, s_ki, s_ab, s_cd;
    const double *boys_tab;
    const uint32_t *rlut;                // [2*N~(24)]: recursion neighbours, packed (t,u,v,n)
};

// per-warp shared memory (doubles): R0[N~(L)] R1[N~(L-1)] G0[L+1] PQ[4] half[nhb*ncd]
__host__ __device__ inline int warp_smem_doubles(int L, int nhb, int ncd) {
    auto even = [](int x) { return x + (x & 1); };
    return even(nherm(L)) + even(L > 0 ? nherm(L - 1) : 1) + even(L + 1) + 4 + even(nhb * ncd);
}

__global__ void __launch_bounds__(MD_WARP_THREADS) eri_warp_kernel(WarpArgs g) {
    extern __shared__ double sm[];
    __shared__ uint32_t s_w[455];                              // packed (t,u,v,n) of the first N~(12) Hermite triples
    const int L = g.Lb + g.Lk, nhb = nherm(g.Lb), nhk = nherm(g.Lk);
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5, nwarp = MD_WARP_THREADS / 32;
    const uint2 *lut = (const uint2 *)g.rlut;
    for (int e = threadIdx.x; e < nherm(L); e += MD_WARP_THREADS) s_w[e] = __ldg(&lut[e].y);
    __syncthreads();
    auto even = [](int x) { return x + (x & 1); };
    const int rs0 = even(nherm(L)), rs1 = even(L > 0 ? nherm(L - 1) : 1);
    double *R0 = sm + (size_t)warp * warp_smem_doubles(L, nhb, g.ncd);
    double *R1 = R0 + rs0, *G0 = R1 + rs1, *PQ = G0 + even(L + 1), *half = PQ + 4;

    for (long long q = (long long)blockIdx.x * nwarp + warp; q < g.nq; q += (long long)gridDim.x * nwarp) {
        long long bi, ki;
        if (g.qidx) { bi = g.qidx[2 * q]; ki = g.qidx[2 * q + 1]; }
        else { bi = q / g.nket; ki = q % g.nket; }
        double *out = g.out + q * g.s_q + bi * g.s_bi + ki * g.s_ki;
        for (int kb = 0; kb < g.Kbra; ++kb) {
            const double *rb = g.rec_bra + (bi * g.Kbra + kb) * g.stride_bra;
            for (int kk = 0; kk < g.Kket; ++kk) {
                const double *rk = g.rec_ket + (ki * g.Kket + kk) * g.stride_ket;
                // S2: [0]^(m), one order per lane                                      (Eqs. 21-23)
                __syncwarp();
                if (lane <= L) {
                    const double p = __ldg(rb), qq = __ldg(rk);
                    const double X = __ldg(rb + 1) - __ldg(rk + 1), Y = __ldg(rb + 2) - __ldg(rk + 2), Z = __ldg(rb + 3) - __ldg(rk + 3);
                    const double rho = p * qq / (p + qq);
                    double f = 34.98683665524972497 / (p * qq * sqrt(p + qq)) * boys_single(lane, rho * (X * X + Y * Y + Z * Z), g.boys_tab);
                    const double m2r = -2.0 * rho;
                    for (int i = 0; i < lane; ++i) f *= m2r;
                    G0[lane] = f;
                    if (lane == L) ((L & 1) ? R1 : R0)[0] = f;
                    if (lane == 0) { PQ[0] = X; PQ[1] = Y; PQ[2] = Z; }
                }
                __syncwarp();
                // S3: Eq. 24 level by level, level m from level m+1 (ping-pong, level 0 lands in R0)
                for (int m = L - 1; m >= 0; --m) {
                    const double *old = (m & 1) ? R0 : R1;
                    double *nw = (m & 1) ? R1 : R0;
                    const int ne = nherm(L - m);
                    for (int e = lane; e < ne; e += 32) {
                        const uint32_t w = __ldg(&lut[e].x);
                        double val;
                        if (e == 0) val = G0[m];
                        else {
                            val = PQ[w >> 24 & 3] * old[w & 0xfff];
                            const int cf = w >> 26;
                            if (cf) val = fma((double)cf, old[w >> 12 & 0xfff], val);
                        }
                        nw[e] = val;
                    }
                    __syncwarp();
                }
                // S4a: [p~|cd] (+)= sum_q~ [p~+q~]^(0) Hk[q~][cd]            (Eqs. 19, 25; the sign is in Hk)
                // With enough Hermite rows the lanes own rows p~ and block 8 columns cd in registers: one gathered
                // [p~+q~] feeds 8 FMAs and the Hk loads are warp-wide broadcasts; else one (p~, cd) element per lane.
                const double *Hk = rk + 4;
                if (nhb >= 16 && g.ncd >= 4) {
                    // tasks (row p~, chunk of 8 columns) are dealt to the lanes together: 35 rows x 2 chunks take 3 rounds, not 4
                    const int nchunk = (g.ncd + 7) >> 3;
                    for (int task = lane; task < nhb * nchunk; task += 32) {
                        {
                            const int ch = task / nhb, p = task - ch * nhb, cd0 = ch << 3;
                            const int nc = min(8, g.ncd - cd0);
                            const uint32_t wp = s_w[p];
                            double acc[8];
#pragma unroll
                            for (int c = 0; c < 8; ++c) acc[c] = 0.0;
                            for (int iq = g.kq0; iq < nhk; ++iq) {
                                const double r = R0[herm_index_packed(wp + s_w[iq])];
                                const double *hk = Hk + (long long)iq * g.ncd + cd0;
#pragma unroll
                                for (int c = 0; c < 8; ++c)
                                    if (c < nc) acc[c] = fma(r, __ldg(hk + c), acc[c]);
                            }
                            double *h = half + p * g.ncd + cd0;
#pragma unroll
                            for (int c = 0; c < 8; ++c)
                                if (c < nc) { if (kk == 0) h[c] = acc[c]; else h[c] += acc[c]; }
                        }
                    }
                } else {
                    for (int it = lane; it < nhb * g.ncd; it += 32) {
                        const int p = it / g.ncd, cd = it - p * g.ncd;
                        const uint32_t wp = s_w[p];
                        double a = 0.0;
                        for (int iq = g.kq0; iq < nhk; ++iq)
                            a = fma(R0[herm_index_packed(wp + s_w[iq])], __ldg(Hk + (long long)iq * g.ncd + cd), a);
                        if (kk == 0) half[it] = a; else half[it] += a;
                    }
                }
            }
            __syncwarp();
            // S4b: [ab|cd] (+)= sum_p~ Hb[p~][ab] [p~|cd]                    (Eq. 26); S5 is folded into Hb, Hk
            const double *Hb = rb + 4;
            if (g.nab >= 16 && g.ncd >= 4) {                   // a lane owns (ab, chunk of 8 columns cd) in registers
                const int nchunk = (g.ncd + 7) >> 3;
                for (int task = lane; task < g.nab * nchunk; task += 32) {
                    {
                        const int ch = task / g.nab, ab = task - ch * g.nab, cd0 = ch << 3;
                        const int nc = min(8, g.ncd - cd0);
                        double acc[8];
#pragma unroll
                        for (int c = 0; c < 8; ++c) acc[c] = 0.0;
                        for (int p = 0; p < nhb; ++p) {
                            const double hb = __ldg(Hb + (long long)p * g.nab + ab);
                            const double *h = half + p * g.ncd + cd0;
#pragma unroll
                            for (int c = 0; c < 8; ++c)
                                if (c < nc) acc[c] = fma(hb, h[c], acc[c]);
                        }
                        double *o = out + ab * g.s_ab + cd0 * g.s_cd;
#pragma unroll
                        for (int c = 0; c < 8; ++c)
                            if (c < nc) { if (kb == 0) o[c * g.s_cd] = acc[c]; else o[c * g.s_cd] += acc[c]; }
                    }
                }
            } else {
                for (int it = lane; it < g.nab * g.ncd; it += 32) {
                    const int ab = it / g.ncd, cd = it - ab * g.ncd;
                    double a = 0.0;
                    for (int p = 0; p < nhb; ++p) a = fma(__ldg(Hb + (long long)p * g.nab + ab), half[p * g.ncd + cd], a);
                    double *o = out + ab * g.s_ab + cd * g.s_cd;
                    if (kb == 0) *o = a; else *o += a;
                }
            }
        }
    }
}

}  // namespace mdb
