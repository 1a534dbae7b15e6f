// fused_kernel.cuh -- compile-time-l fused kernel: ONE launch runs S1-S5 for a class (la lb|lc ld).
//
// A CTA of 256 threads works on NQ quartets at a time; every per-quartet quantity lives in
// shared memory or registers (no HBM traffic except the shell data in and the integrals out,
// PAPER.md:143-146).  Unlike the paper's dense H formulation (Eqs. 17, 25, 26), the two
// Hermite->AO contractions run over the SPARSE Cartesian expansion
//     E^{cd}_{q~} = E^{t'}_{cx dx} E^{u'}_{cy dy} E^{v'}_{cz dz},  non-zero only for t' <= cx+dx, ..   (Eqs. 7, 14)
// and the solid-harmonic matrices (Eq. 16) are applied afterwards with their zeros skipped.
// Both are the same sums as Eqs. 25-26 in another order; for independent quartets this needs
// about 2.2x fewer FMAs for (dd|dd) than building dense solid H per pair.
//
// Phases per primitive quartet (kb, kk), each separated by a CTA barrier:
//   P1  thread (quartet, axis): 1-D tables E^t_{ij} in registers -> shared          (Eqs. 9,10,13,14)
//   P2  thread (quartet, m): [0]^(m) from the per-order Boys Taylor table            (Eqs. 21-23)
//       thread (quartet, cd): the list of E^{cd}_{q~} products, with (-1)^{|q~|} of Eq. 19
//   P3  [r]^(m) levels m = L-1..0 over compact ping-pong buffers; level 0 lands in a cube  (Eq. 24)
//   P4  thread (quartet, p~): [p~|cd] += sum_q~ E^{cd}_{q~} [p~+q~]^(0)  -- registers  (Eq. 25)
// then per bra primitive: solid transform of cd in registers, [p~|cd] -> shared,
//   P5  thread (quartet, cd): [ab|cd] += sum_p~ E^{ab}_{p~} [p~|cd]       -- registers  (Eq. 26)
// and finally the solid transform of ab in registers and the store.
#pragma once
#include "boys.cuh"
#include "fused_tables.cuh"

namespace mdb {

#define MD_FUSED_THREADS 256

struct FusedArgs {
    PairView bra, ket;            // shells already in the kernel's (canonical) order
    int bra_swap, ket_swap;       // 1: the pair index columns are (b,a) / (d,c)
    const int32_t *qidx;
    long long nq, nket;
    double *out;
    long long s_q, s_bi, s_ki;    // quartet base = q*s_q + bi*s_bi + ki*s_ki
    long long sa, sb, sc, sd;     // component strides of the kernel's four shells
    const double *boys_tab;
    const uint32_t *rlut;         // [2*N~(24)]: R-recursion neighbours and packed (t,u,v)
    // Exchange digestion (Eq. 32, K_bc += sum_ad [ab|cd] D_ad): when dg_K != nullptr nothing is stored to `out`;
    // each thread contracts its integrals with D and adds into K.  dg_off[s] = AO offset of every shell of the kernel's
    // shell s (kernel order, i.e. after the canonical swaps); D and K are [dg_n][dg_n], row-major.
    double *dg_K = nullptr;
    const double *dg_D = nullptr;
    const int32_t *dg_off[4] = {nullptr, nullptr, nullptr, nullptr};
    long long dg_n = 0;
};

template <int LA, int LB, int LC, int LD, bool PURE>
struct FusedCfg {
    static constexpr int Lb = LA + LB, Lk = LC + LD, L = Lb + Lk, S = L + 1;
    static constexpr int NHB = nherm(Lb), NHK = nherm(Lk), NHL = nherm(L);
    static constexpr int NCA = ncart(LA), NCB = ncart(LB), NCC = ncart(LC), NCD = ncart(LD);
    static constexpr int NAO = ncomp(LA, PURE), NBO = ncomp(LB, PURE), NCO = ncomp(LC, PURE), NDO = ncomp(LD, PURE);
    static constexpr int NAB_C = NCA * NCB, NCD_C = NCC * NCD, NAB_O = NAO * NBO, NCD_O = NCO * NDO;
    static constexpr int NPB = ProdCount<LA, LB>::value(), NPK = ProdCount<LC, LD>::value();
    static constexpr int W = NHB > NCD_O ? NHB : NCD_O;
    static constexpr int NQ = MD_FUSED_THREADS / W > 0 ? MD_FUSED_THREADS / W : 1;
    static constexpr int HS = NCD_O | 1;                       // odd row stride of [p~|cd]: conflict-free
    // per-quartet shared memory, in doubles
    static constexpr int E1B = 3 * (LA + 1) * (LB + 1) * (Lb + 1), E1K = 3 * (LC + 1) * (LD + 1) * (Lk + 1);
    static constexpr int even(int x) { return x + (x & 1); }
    static constexpr int O_HDR = 0;                            // 16 doubles
    static constexpr int O_G0 = 16;                            // [L+1]
    static constexpr int O_E1B = O_G0 + even(S);
    static constexpr int O_E1K = O_E1B + even(E1B);
    static constexpr int O_PROD = O_E1K + even(E1K);           // max(NPB, NPK)
    static constexpr int O_RB = O_PROD + even(NPB > NPK ? NPB : NPK);   // 2 x N~(L-1) ping-pong
    static constexpr int NRB = even(L > 0 ? nherm(L - 1) : 1);
    static constexpr int O_U = O_RB + 2 * NRB;                 // union { cube[S^3], half[NHB][HS] }
    static constexpr int NU = even(S * S * S > NHB * HS ? S * S * S : NHB * HS);
    static constexpr int PERQ = O_U + NU;
    static constexpr int LUT_D = even(NHL);                    // 2 uint32 per Hermite entry = NHL doubles
    static constexpr size_t SMEM = 8 * (size_t)(LUT_D + 4 * NQ / 2 + 2 + NQ * PERQ);
    static_assert(W <= MD_FUSED_THREADS, "class too large for the fused kernel");
};

// hdr slots
enum { H_P = 0, H_PX = 1, H_CAB = 4, H_Q = 5, H_QX = 6, H_CCD = 9, H_PQX = 10 };

// One Cartesian axis of the two-centre table (Eqs. 9, 10, 13, 14), recursion in registers.
// Writes E[(i*(L2+1)+j)*(L1+L2+1)+t].
template <int L1, int L2>
__device__ __forceinline__ void axis_table(double za, double zb, double xab, double *E) {
    constexpr int NT = L1 + L2 + 1;
    const double p = za + zb, ip = 1.0 / p, h = 0.5 * ip;
    const double xpa = -zb * xab * ip, xpb = za * xab * ip;
    double e[L1 + 1][L2 + 1][NT];
#pragma unroll
    for (int i = 0; i <= L1; ++i)
#pragma unroll
        for (int j = 0; j <= L2; ++j)
#pragma unroll
            for (int t = 0; t < NT; ++t) e[i][j][t] = 0.0;
    e[0][0][0] = exp(-za * zb * ip * xab * xab);
#pragma unroll
    for (int j = 0; j < L2; ++j)
#pragma unroll
        for (int t = 0; t <= j + 1; ++t) {
            double v = xpb * e[0][j][t];
            if (t > 0) v = fma(h, e[0][j][t - 1], v);
            if (t < j) v = fma((double)(t + 1), e[0][j][t + 1], v);
            e[0][j + 1][t] = v;
        }
#pragma unroll
    for (int i = 0; i < L1; ++i)
#pragma unroll
        for (int j = 0; j <= L2; ++j)
#pragma unroll
            for (int t = 0; t <= i + j + 1; ++t) {
                double v = xpa * e[i][j][t];
                if (t > 0) v = fma(h, e[i][j][t - 1], v);
                if (t < i + j) v = fma((double)(t + 1), e[i][j][t + 1], v);
                e[i + 1][j][t] = v;
            }
#pragma unroll
    for (int i = 0; i <= L1; ++i)
#pragma unroll
        for (int j = 0; j <= L2; ++j)
#pragma unroll
            for (int t = 0; t <= i + j; ++t) E[(i * (L2 + 1) + j) * NT + t] = e[i][j][t];
}

// P1 for one side: threads (quartet j, axis) fill the tables and the pair header.
template <int L1, int L2>
__device__ __forceinline__ void pair_phase(const PairView &pv, const int *sidx, int col, int k1, int k2, int nqg,
                                           double *qsm, int perq, int o_e1, int o_hdr, int tid) {
    constexpr int ESZ = (L1 + 1) * (L2 + 1) * (L1 + L2 + 1);
    for (int it = tid; it < 3 * nqg; it += MD_FUSED_THREADS) {
        const int j = it / 3, ax = it % 3;
        const long long i1 = sidx[4 * j + col], i2 = sidx[4 * j + col + 1];
        const int K1 = pv.a.K, K2 = pv.b.K;
        const double za = pv.a.exps[i1 * K1 + k1], A = pv.a.center[3 * i1 + ax];
        double zb = 0.0, B = A;
        if (!pv.single) { zb = pv.b.exps[i2 * K2 + k2]; B = pv.b.center[3 * i2 + ax]; }
        double *q = qsm + (size_t)j * perq;
        axis_table<L1, L2>(za, zb, A - B, q + o_e1 + ax * ESZ);
        const double p = za + zb;
        q[o_hdr + 1 + ax] = (za * A + zb * B) / p;
        if (ax == 0) {
            q[o_hdr] = p;
            q[o_hdr + 4] = pv.a.coefs[i1 * K1 + k1] * (pv.single ? 1.0 : pv.b.coefs[i2 * K2 + k2]);
        }
    }
}

// The list of E products of one side (consumed in ProdList order), optionally with (-1)^{t+u+v}.
template <int L1, int L2, bool SIGN>
__device__ __forceinline__ void prod_phase(int nqg, double *qsm, int perq, int o_e1, int o_coef, int o_prod, int tid) {
    constexpr int NC1 = ncart(L1), NC2 = ncart(L2), NCOMP = NC1 * NC2, NT = L1 + L2 + 1;
    constexpr int ESZ = (L1 + 1) * (L2 + 1) * NT;
    const short *start = d_prod_start<L1, L2>.start;
    for (int it = tid; it < nqg * NCOMP; it += MD_FUSED_THREADS) {
        const int j = it / NCOMP, comp = it % NCOMP, c = comp / NC2, d = comp % NC2;
        int ax, ay, az, bx, by, bz;
        unpack_tuv(c_herm[nherm(L1 - 1) + c], ax, ay, az);
        unpack_tuv(c_herm[nherm(L2 - 1) + d], bx, by, bz);
        double *q = qsm + (size_t)j * perq;
        const double *Ex = q + o_e1 + (ax * (L2 + 1) + bx) * NT;
        const double *Ey = q + o_e1 + ESZ + (ay * (L2 + 1) + by) * NT;
        const double *Ez = q + o_e1 + 2 * ESZ + (az * (L2 + 1) + bz) * NT;
        const double coef = q[o_coef];
        double *dst = q + o_prod + start[comp];
        for (int t = 0; t <= ax + bx; ++t) {
            const double et = coef * Ex[t];
            for (int u = 0; u <= ay + by; ++u) {
                const double eu = et * Ey[u];
                for (int v = 0; v <= az + bz; ++v) {
                    double val = eu * Ez[v];
                    if (SIGN && ((t + u + v) & 1)) val = -val;
                    *dst++ = val;
                }
            }
        }
    }
}

// In-register Cartesian -> solid transform of a [N1c][N2c] block to [N1o][N2o] (Eq. 16, zeros skipped).
template <int L1, int L2, bool PURE>
__device__ __forceinline__ void solid2(const double (&in)[ncart(L1) * ncart(L2)],
                                       double (&out)[ncomp(L1, PURE) * ncomp(L2, PURE)]) {
    constexpr int N1 = ncart(L1), N2 = ncart(L2);
    if constexpr (!PURE) {
#pragma unroll
        for (int i = 0; i < N1 * N2; ++i) out[i] = in[i];
    } else {
        constexpr int M1 = nsolid(L1), M2 = nsolid(L2);
        constexpr SolidTab<L1> C1{};
        constexpr SolidTab<L2> C2{};
        double t1[N1 * M2];
#pragma unroll
        for (int a = 0; a < N1; ++a)
#pragma unroll
            for (int m = 0; m < M2; ++m) {
                double s = 0.0;
#pragma unroll
                for (int b = 0; b < N2; ++b)
                    if (C2.c[m][b] != 0.0) s = fma(C2.c[m][b], in[a * N2 + b], s);
                t1[a * M2 + m] = s;
            }
#pragma unroll
        for (int ma = 0; ma < M1; ++ma)
#pragma unroll
            for (int m = 0; m < M2; ++m) {
                double s = 0.0;
#pragma unroll
                for (int a = 0; a < N1; ++a)
                    if (C1.c[ma][a] != 0.0) s = fma(C1.c[ma][a], t1[a * M2 + m], s);
                out[ma * M2 + m] = s;
            }
    }
}

template <int LA, int LB, int LC, int LD, bool PURE>
__global__ void __launch_bounds__(MD_FUSED_THREADS) fused_kernel(FusedArgs g) {
    using C = FusedCfg<LA, LB, LC, LD, PURE>;
    constexpr int L = C::L, S = C::S, NQ = C::NQ, PERQ = C::PERQ;
    extern __shared__ double sm[];
    uint32_t *lut = (uint32_t *)sm;                         // [2*NHL]
    int *sidx = (int *)(sm + C::LUT_D);                     // [NQ][4] shell indices a,b,c,d
    double *qsm = sm + C::LUT_D + 4 * NQ / 2 + 2;
    const int tid = threadIdx.x;

    for (int e = tid; e < 2 * C::NHL; e += MD_FUSED_THREADS) lut[e] = g.rlut[e];

    // fixed roles
    const int j1 = tid / C::NHB, ip = tid % C::NHB;         // P4: (quartet, p~)
    const int j2 = tid / C::NCD_O, icd = tid % C::NCD_O;    // P5: (quartet, output cd)
    const int Ka = g.bra.a.K, Kb = g.bra.single ? 1 : g.bra.b.K;
    const int Kc = g.ket.a.K, Kd = g.ket.single ? 1 : g.ket.b.K;
    __syncthreads();
    int cube_ip;
    {
        int t, u, v;
        unpack_tuv(lut[2 * ip + 1], t, u, v);
        cube_ip = (t * S + u) * S + v;
    }

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
            sidx[4 * tid] = (int)ia; sidx[4 * tid + 1] = (int)ib; sidx[4 * tid + 2] = (int)ic; sidx[4 * tid + 3] = (int)id;
        }
        __syncthreads();

        double oacc[C::NAB_C];
#pragma unroll
        for (int i = 0; i < C::NAB_C; ++i) oacc[i] = 0.0;

        for (int kb = 0; kb < Ka * Kb; ++kb) {
            pair_phase<LA, LB>(g.bra, sidx, 0, kb / Kb, kb % Kb, nqg, qsm, PERQ, C::O_E1B, H_P, tid);
            double hacc[C::NCD_C];
#pragma unroll
            for (int i = 0; i < C::NCD_C; ++i) hacc[i] = 0.0;

            for (int kk = 0; kk < Kc * Kd; ++kk) {
                pair_phase<LC, LD>(g.ket, sidx, 2, kk / Kd, kk % Kd, nqg, qsm, PERQ, C::O_E1K, H_Q, tid);
                __syncthreads();                             // tables ready; previous P4 finished everywhere
                // P2a: [0]^(m)
                for (int it = tid; it < nqg * S; it += MD_FUSED_THREADS) {
                    const int j = it / S, m = it % S;
                    double *q = qsm + (size_t)j * PERQ;
                    const double p = q[H_P], qq = q[H_Q];
                    const double X = q[H_PX] - q[H_QX], Y = q[H_PX + 1] - q[H_QX + 1], Z = q[H_PX + 2] - q[H_QX + 2];
                    const double rho = p * qq / (p + qq);
                    const double T = rho * (X * X + Y * Y + Z * Z);
                    double f = 34.98683665524972497 / (p * qq * sqrt(p + qq)) * boys_single(m, T, g.boys_tab);
                    const double m2r = -2.0 * rho;
                    for (int i = 0; i < m; ++i) f *= m2r;
                    q[C::O_G0 + m] = f;
                    if (m == L) q[C::O_RB + (L & 1) * C::NRB] = f;     // level L = { [0]^(L) }
                    if (m == 0) { q[H_PQX] = X; q[H_PQX + 1] = Y; q[H_PQX + 2] = Z; }
                }
                // P2b: ket E products, sign of Eq. 19 folded in
                prod_phase<LC, LD, true>(nqg, qsm, PERQ, C::O_E1K, H_CCD, C::O_PROD, tid);
                __syncthreads();
                // P3: Eq. 24 level by level; level m reads buffer (m+1)&1, writes m&1; level 0 -> cube
                if constexpr (L == 0) {
                    if (tid < nqg) qsm[(size_t)tid * PERQ + C::O_U] = qsm[(size_t)tid * PERQ + C::O_G0];
                    __syncthreads();
                }
#pragma unroll
                for (int m = L - 1; m >= 0; --m) {
                    constexpr int dummy = 0; (void)dummy;
                    const int ne = nherm(L - m);
                    for (int it = tid; it < nqg * ne; it += MD_FUSED_THREADS) {
                        const int j = it / ne, e = it % ne;
                        double *q = qsm + (size_t)j * PERQ;
                        const double *old = q + C::O_RB + ((m + 1) & 1) * C::NRB;
                        const uint32_t w = lut[2 * e];
                        double val;
                        if (e == 0) val = q[C::O_G0 + m];
                        else {
                            val = q[H_PQX + (w >> 24 & 3)] * old[w & 0xfff];
                            const int cf = w >> 26;
                            if (cf) val = fma((double)cf, old[w >> 12 & 0xfff], val);
                        }
                        if (m > 0) q[C::O_RB + (m & 1) * C::NRB + e] = val;
                        else {
                            int t, u, v;
                            unpack_tuv(lut[2 * e + 1], t, u, v);
                            q[C::O_U + (t * S + u) * S + v] = val;
                        }
                    }
                    __syncthreads();
                }
                // P4: [p~|cd] += sum E^{cd}_{q~} R[cube(p~) + cube(q~)]
                if (j1 < nqg) {
                    const double *q = qsm + (size_t)j1 * PERQ;
                    const double *Rb = q + C::O_U + cube_ip;
                    const double2 *ep = (const double2 *)(q + C::O_PROD);
                    constexpr ProdList<LC, LD, S> PK{};
#pragma unroll
                    for (int i = 0; i < PK.N; i += 2) {
                        const double2 e2 = ep[i / 2];
                        hacc[PK.comp[i]] = fma(e2.x, Rb[PK.off[i]], hacc[PK.comp[i]]);
                        if (i + 1 < PK.N) hacc[PK.comp[i + 1]] = fma(e2.y, Rb[PK.off[i + 1]], hacc[PK.comp[i + 1]]);
                    }
                }
            }
            // ket solid transform in registers, then [p~|cd] -> shared (over the cube) and bra products
            double h2[C::NCD_O];
            solid2<LC, LD, PURE>(hacc, h2);
            __syncthreads();                                 // everyone is done reading the cube / ket products
            if (j1 < nqg) {
                double *half = qsm + (size_t)j1 * PERQ + C::O_U + ip * C::HS;
#pragma unroll
                for (int i = 0; i < C::NCD_O; ++i) half[i] = h2[i];
            }
            prod_phase<LA, LB, false>(nqg, qsm, PERQ, C::O_E1B, H_CAB, C::O_PROD, tid);
            __syncthreads();
            // P5: [ab|cd] += sum E^{ab}_{p~} [p~|cd]
            if (j2 < nqg) {
                const double *q = qsm + (size_t)j2 * PERQ;
                const double *half = q + C::O_U + icd;
                double hv[C::NHB];
#pragma unroll
                for (int i = 0; i < C::NHB; ++i) hv[i] = half[i * C::HS];
                const double2 *ep = (const double2 *)(q + C::O_PROD);
                constexpr ProdList<LA, LB, 0> PB{};
#pragma unroll
                for (int i = 0; i < PB.N; i += 2) {
                    const double2 e2 = ep[i / 2];
                    oacc[PB.comp[i]] = fma(e2.x, hv[PB.off[i]], oacc[PB.comp[i]]);
                    if (i + 1 < PB.N) oacc[PB.comp[i + 1]] = fma(e2.y, hv[PB.off[i + 1]], oacc[PB.comp[i + 1]]);
                }
            }
            // the next kb (or group) starts with pair_phase + barrier before shared memory is rewritten
        }
        // bra solid transform and store
        if (j2 < nqg) {
            double o2[C::NAB_O];
            solid2<LA, LB, PURE>(oacc, o2);
            const long long q = q0 + j2;
            long long bi, ki;
            if (g.qidx) { bi = g.qidx[2 * q]; ki = g.qidx[2 * q + 1]; }
            else { bi = q / g.nket; ki = q % g.nket; }
            if (g.dg_K) {
                // In caller order K[b][c] += [ab|cd] D[a][d]; the kernel's shells may be (b,a) and/or (d,c).  This thread
                // holds one (c',d') column and all (a',b'): the D-side bra index is summed in registers, one atomic per K row.
                long long ia = bi, ib = bi, ic = ki, id = ki;
                if (g.bra.idx) { ia = g.bra.idx[2 * bi + g.bra_swap]; ib = g.bra.idx[2 * bi + 1 - g.bra_swap]; }
                if (g.ket.idx) { ic = g.ket.idx[2 * ki + g.ket_swap]; id = g.ket.idx[2 * ki + 1 - g.ket_swap]; }
                const long long oa = g.dg_off[0][ia], ob = g.dg_off[1][ib];
                const long long oc = g.dg_off[2][ic] + icd / C::NDO, od = g.dg_off[3][id] + icd % C::NDO;
                const long long kcol = g.ket_swap ? od : oc, dcol = g.ket_swap ? oc : od;
                if (!g.bra_swap) {                                   // a' = a (D row), b' = b (K row)
#pragma unroll
                    for (int b = 0; b < C::NBO; ++b) {
                        double s = 0.0;
#pragma unroll
                        for (int a = 0; a < C::NAO; ++a) s = fma(o2[a * C::NBO + b], g.dg_D[(oa + a) * g.dg_n + dcol], s);
                        atomicAdd(g.dg_K + (ob + b) * g.dg_n + kcol, s);
                    }
                } else {                                             // a' = b (K row), b' = a (D row)
#pragma unroll
                    for (int a = 0; a < C::NAO; ++a) {
                        double s = 0.0;
#pragma unroll
                        for (int b = 0; b < C::NBO; ++b) s = fma(o2[a * C::NBO + b], g.dg_D[(ob + b) * g.dg_n + dcol], s);
                        atomicAdd(g.dg_K + (oa + a) * g.dg_n + kcol, s);
                    }
                }
            } else {
            double *o = g.out + q * g.s_q + bi * g.s_bi + ki * g.s_ki + (icd / C::NDO) * g.sc + (icd % C::NDO) * g.sd;
#pragma unroll
            for (int a = 0; a < C::NAO; ++a)
#pragma unroll
                for (int b = 0; b < C::NBO; ++b) o[a * g.sa + b * g.sb] = o2[a * C::NBO + b];
            }
        }
    }
}

}  // namespace mdb
