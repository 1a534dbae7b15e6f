// eri3s.cuh -- 3-center integrals (ab|X) with la, lb <= 3: ONE WARP per triplet, sparse Cartesian bra, no dense H.
//
// BASELINE configs[2] (density-fitting shape: la, lb in 0..3, K = 1..4 per bra shell, lX in 0..6).  With a single shell on the
// ket side N_cd = 2 lX + 1 is small, and forming the dense bra matrix H[p~][ab] per primitive pair (Eq. 17: about 2 N~ N_ab n_c
// FMAs) costs ten times the contraction it feeds.  This kernel applies the bra expansion in its factorised Cartesian form
// instead (Eqs. 7, 9, 10, 13, 14: E^{ab}_{p~} = E^t_{ax bx} E^u_{ay by} E^v_{az bz}, zero for t > ax+bx ..):
//   per bra primitive pair   three 1-D tables by the warp (lane = t);
//   per X primitive          F_m (one order per lane), [r~]^(0) level by level (Eqs. 21-24) in the warp's shared memory,
//                            G[p~][c] += sum_q~ H_X[q~][c] [p~+q~]^(0)   (Eqs. 19, 25; solid X by the Hobson form: only |q~| = lX);
//   per bra primitive pair   acc[a b][c] += c_a c_b sum_{tuv in the box of (a,b)} E^t E^u E^v G[tuv][c]   (Eq. 26), lane = (a,b);
//   per triplet              Cartesian -> solid on a and b (Eq. 16) through shared memory, one contiguous coalesced store.
// Everything between the shell data and the result stays in registers and the warp's slice of shared memory
// (PAPER.md:143-146); there is no CTA barrier and no scratch.
#pragma once
#include "hl.cuh"

namespace mdb {

struct Eri3sArgs {
    PairView bra;
    ShellView X;                          // the one-centre ket shell, or shell c of a two-centre ket (c, s)
    ShellView D;                          // two-centre ket: its s shell d
    const int32_t *kidx;                  // two-centre ket: pair list (c, d) or nullptr
    int KD, lD, swap;                     // lD: angular momentum of d (two-centre ket); swap = 1: the kernel's bra is the CALLER's ket (index columns and output strides swapped)
    long long s_t, s_ab, s_c;             // output strides (doubles) of the triplet / quartet, the ab block index, the c index
    int pure, la, lb, lX, Ka, Kb, KX;
    int nca, ncb, nXc, nhb, L;            // Cartesian counts of a, b; components of X in the result; N~(la+lb); la+lb+lX
    const int32_t *tidx;                  // [n][2] (bra pair, X shell) or nullptr: product, X fastest
    long long nt, nX;
    double *out;                          // [t][a][b][c]
    const double *boys_tab;
    const uint32_t *rlut;
    int warps, per_warp;                  // shared-memory doubles per warp
    int o_r0, o_r1, o_g, o_acc, o_e, o_ex, o_g0;   // offsets inside a warp's slice
};

// NXC = components of X in the result (2 lX + 1, or the Cartesian count), a compile-time constant so that the two hot loops
// (Hobson G build, bra box loop) unroll exactly: with a run-time count every multiply-add carried a compare and its own
// 8-byte shared-memory load (34 % + 28 % of the stall samples of (ff|f) K = 4, profiles/r02_eri3s.md).
// MODE 0: one-centre solid X (Hobson form); 1: one-centre Cartesian X; 2: two-centre ket (c, d) of a 4-center class -- G is
// built in the Cartesian components (c, d) from the three 1-D tables of the ket pair (Eqs. 9, 10, 13), NXC = ncart(lc) ncart(ld)
// columns, and the solid transforms of d and c (Eq. 16), if asked for, are two more passes at the end.
template <int NXC, int MODE>
__global__ void __launch_bounds__(256) eri3s_kernel(Eri3sArgs g) {
    constexpr bool PURE = MODE == 0, TWO = MODE == 2;
    extern __shared__ double sm[];
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    // CTA-wide constants: Hermite triples and the transposed Cartesian->solid tables of a, b, X
    uint32_t *s_herm = (uint32_t *)sm;                               // nherm(12) words
    double *CT = sm + 228;                                           // 4 x 28 x MD_HL_CSTR
    const int ls[4] = {g.la, g.lb, g.lX, MODE == 2 ? g.lD : 0};
    if (blockDim.x == 256) hl_stage_tables<256>(s_herm, nherm(g.L), CT, ls);
    else hl_stage_tables<128>(s_herm, nherm(g.L), CT, ls);
    const int CTS = 28 * MD_HL_CSTR;
    uint16_t *cube = (uint16_t *)(sm + 228 + 4 * CTS);               // (t,u,v) -> position in the degree-sorted list, t,u,v <= la+lb
    {
        const int S = g.la + g.lb + 1;
        for (int i = threadIdx.x; i < S * S * S; i += blockDim.x) {
            const int t = i / (S * S), u = i / S % S, v = i % S;
            cube[i] = t + u + v < S ? (uint16_t)herm_index(t, u, v) : (uint16_t)0;
        }
    }
    __syncthreads();
    if (warp >= g.warps) return;
    const double *CaT = CT, *CbT = CT + CTS, *CxT = CT + 2 * CTS;
    double *W = sm + 228 + 4 * CTS + 88 + (size_t)warp * g.per_warp;
    double *R0 = W + g.o_r0, *R1 = W + g.o_r1, *G = W + g.o_g, *acc = W + g.o_acc, *E = W + g.o_e, *EX = W + g.o_ex, *G0 = W + g.o_g0;
    const uint2 *lut = (const uint2 *)g.rlut;
    const int la = g.la, lb = g.lb, lX = g.lX, Lb = la + lb, L = g.L, nt = Lb + 1;
    constexpr int nXc = NXC;
    // columns a lane keeps in registers per pass of the bra box loop: all of them up to 12, else a divisor, else 7
    constexpr int CW = nXc <= 12 ? nXc : nXc % 12 == 0 ? 12 : nXc % 10 == 0 ? 10 : nXc % 9 == 0 ? 9 : nXc == 15 ? 8 : 7;
    const int nca = g.nca, ncb = g.ncb, nhb = g.nhb, nab_c = nca * ncb;
    const int esz = (la + 1) * (lb + 1) * nt;
    const uint32_t *ca = s_herm + nherm(la - 1), *cb = s_herm + nherm(lb - 1), *cx = s_herm + nherm(lX - 1);
    const int ncx = ncart(lX), nlow = nherm(lX - 1);
    const int lD = TWO ? g.lD : 0, ncdd = ncart(lD), ntk = lX + lD + 1, eszk = (lX + 1) * (lD + 1) * ntk;   // ket pair tables E[(i (lD+1) + j) ntk + t]
    const uint32_t *cdl = s_herm + nherm(lD - 1);
    const double *CdT = CT + 3 * CTS;
    const long long wstride = (long long)gridDim.x * g.warps;

    for (long long t = (long long)blockIdx.x * g.warps + warp; t < g.nt; t += wstride) {
        long long bi, xi;
        if (g.tidx) { bi = g.tidx[2 * t + g.swap]; xi = g.tidx[2 * t + 1 - g.swap]; }
        else {
            const long long b0 = t / g.nX, k0 = t % g.nX;            // the caller's (bra, ket) of product entry t
            bi = g.swap ? k0 : b0; xi = g.swap ? b0 : k0;
        }
        long long ia = bi, ib = bi, id = xi;
        if (g.bra.idx) { ia = g.bra.idx[2 * bi]; ib = g.bra.idx[2 * bi + 1]; }
        if (TWO && g.kidx) { id = g.kidx[2 * xi + 1]; xi = g.kidx[2 * xi]; }
        double A[3], B[3], Xc[3], Dc[3];
#pragma unroll
        for (int x = 0; x < 3; ++x) {
            A[x] = g.bra.a.center[3 * ia + x]; B[x] = g.bra.b.center[3 * ib + x]; Xc[x] = g.X.center[3 * xi + x];
            Dc[x] = TWO ? g.D.center[3 * id + x] : Xc[x];
        }
        for (int i = lane; i < nab_c * nXc; i += 32) acc[i] = 0.0;
        for (int kab = 0; kab < g.Ka * g.Kb; ++kab) {
            const int ka = kab / g.Kb, kb = kab - ka * g.Kb;
            const double za = g.bra.a.exps[ia * g.Ka + ka], zb = g.bra.b.exps[ib * g.Kb + kb];
            const double cab = g.bra.a.coefs[ia * g.Ka + ka] * g.bra.b.coefs[ib * g.Kb + kb];
            const double p = za + zb;
            __syncwarp();                                            // the previous primitive is done with E and G
#pragma unroll
            for (int x = 0; x < 3; ++x) hl_e_axis_warp(la, lb, za, zb, A[x] - B[x], E + x * esz, lane);
            for (int i = lane; i < nhb * nXc; i += 32) G[i] = 0.0;
            double PQ[3];
#pragma unroll
            for (int x = 0; x < 3; ++x) PQ[x] = (za * A[x] + zb * B[x]) / p - Xc[x];
            for (int kx = 0; kx < g.KX * (TWO ? g.KD : 1); ++kx) {
                double zx, cxc, zc = 0.0, zd = 0.0;                  // zx: the ket exponent q (one-centre: zeta_X)
                if constexpr (TWO) {
                    const int kc = kx / g.KD, kd = kx - kc * g.KD;
                    zc = g.X.exps[xi * g.KX + kc]; zd = g.D.exps[id * g.KD + kd];
                    cxc = g.X.coefs[xi * g.KX + kc] * g.D.coefs[id * g.KD + kd];
                    zx = zc + zd;
#pragma unroll
                    for (int x = 0; x < 3; ++x) PQ[x] = (za * A[x] + zb * B[x]) / p - (zc * Xc[x] + zd * Dc[x]) / zx;
                } else {
                    zx = g.X.exps[xi * g.KX + kx]; cxc = g.X.coefs[xi * g.KX + kx];
                }
                const double rho = p * zx / (p + zx);
                const double T = rho * (PQ[0] * PQ[0] + PQ[1] * PQ[1] + PQ[2] * PQ[2]);
                __syncwarp();
                if (lane <= L) {                                     // [0]^(m) (Eq. 21), one order per lane
                    double f = 34.98683665524972497 * cab * cxc / (p * zx * sqrt(p + zx)) * boys_single(lane, T, g.boys_tab);
                    const double m2r = -2.0 * rho;
                    for (int i = 0; i < lane; ++i) f *= m2r;
                    G0[lane] = f;
                    if (lane == L) ((L & 1) ? R1 : R0)[0] = f;
                }
                if constexpr (TWO) {                                 // the ket pair: E^t_{ij} per axis, exponential included (Eq. 13)
#pragma unroll
                    for (int x = 0; x < 3; ++x) hl_e_axis_warp(lX, lD, zc, zd, Xc[x] - Dc[x], EX + x * eszk, lane);
                } else if (!PURE) hl_e_axis_warp(lX, 0, zx, 0.0, 0.0, EX, lane);   // one-centre table (Eq. 8), the same on the three axes
                __syncwarp();
                for (int m = L - 1; m >= 0; --m) {                   // Eq. 24, level m from level m + 1
                    const int ne = nherm(L - m);
                    const double *old = (m & 1) ? R0 : R1;
                    double *nw = (m & 1) ? R1 : R0;
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
                // G[p~][c] += sum_q~ H_X[q~][c] (-1)^{|q~|} [p~+q~]^(0)
                if constexpr (PURE) {
                    double f = (lX & 1) ? -1.0 : 1.0;                // Hobson: C^l_{m,q~}/(2 zeta)^l on the order-lX Hermites only
                    for (int i = 0; i < lX; ++i) f *= 0.5 / zx;
                    for (int ip = lane; ip < nhb; ip += 32) {          // lane = p~: 13 accumulators, C^{lX}[q~][m] broadcast to the warp
                        const uint32_t wp = s_herm[ip];
                        constexpr int NP = (nXc + 1) / 2;             // coefficient rows are zero-padded to MD_HL_CSTR: 16-byte loads
                        double sacc[2 * NP];
#pragma unroll
                        for (int m = 0; m < 2 * NP; ++m) sacc[m] = 0.0;
                        for (int j = 0; j < ncx; ++j) {
                            const double r = R0[hl_herm_index(wp + cx[j])];
                            const double2 *c = (const double2 *)(CxT + j * MD_HL_CSTR);
#pragma unroll
                            for (int m = 0; m < NP; ++m) {
                                const double2 cc = c[m];
                                sacc[2 * m] = fma(cc.x, r, sacc[2 * m]);
                                sacc[2 * m + 1] = fma(cc.y, r, sacc[2 * m + 1]);
                            }
                        }
                        double *o = G + ip * nXc;
#pragma unroll
                        for (int m = 0; m < nXc; ++m) o[m] = fma(f, sacc[m], o[m]);
                    }
                } else if constexpr (nXc <= 15 || (TWO && nXc != 21 && nXc != 28)) {
                    // The dense table HX[q~][col] = (-1)^{|q~|} E^t E^u E^v of this ket primitive (Eqs. 7, 8, 19; zero where a Hermite
                    // index exceeds the Cartesian sum), then lane = p~ with every column in registers: about three times the
                    // multiply-adds of the sparse walk below, but no per-element box loop and no divergence.  col = c ncart(lD) + d.
                    const int nhx = nherm(lX + lD), exsz = (TWO ? 3 : 1) * eszk;
                    const double *EY = TWO ? EX + eszk : EX, *EZ = TWO ? EX + 2 * eszk : EX;
                    constexpr int NP = (nXc + 1) / 2, HS = 2 * NP;
                    double *HX = EX + exsz + (exsz & 1);
                    for (int i = lane; i < nhx * HS; i += 32) {
                        const int iq = i / HS, c = i - iq * HS;
                        double e3 = 0.0;
                        if (c < nXc) {
                            const int ci = c / ncdd, di = c - ci * ncdd;
                            int ex, ey, ez, dx, dy, dz, t2, u2, v2;
                            unpack_tuv(cx[ci], ex, ey, ez);
                            unpack_tuv(cdl[di], dx, dy, dz);
                            unpack_tuv(s_herm[iq], t2, u2, v2);
                            if (t2 <= ex + dx && u2 <= ey + dy && v2 <= ez + dz) {
                                e3 = EX[(ex * (lD + 1) + dx) * ntk + t2] * EY[(ey * (lD + 1) + dy) * ntk + u2] * EZ[(ez * (lD + 1) + dz) * ntk + v2];
                                if ((t2 + u2 + v2) & 1) e3 = -e3;
                            }
                        }
                        HX[i] = e3;
                    }
                    __syncwarp();
                    for (int ip = lane; ip < nhb; ip += 32) {
                        const uint32_t wp = s_herm[ip];
                        double sacc[HS];
#pragma unroll
                        for (int m = 0; m < HS; ++m) sacc[m] = 0.0;
                        for (int iq = 0; iq < nhx; ++iq) {
                            const double r = R0[hl_herm_index(wp + s_herm[iq])];
                            const double2 *h = (const double2 *)(HX + iq * HS);
#pragma unroll
                            for (int m = 0; m < NP; ++m) {
                                const double2 hh = h[m];
                                sacc[2 * m] = fma(hh.x, r, sacc[2 * m]);
                                sacc[2 * m + 1] = fma(hh.y, r, sacc[2 * m + 1]);
                            }
                        }
                        double *o = G + ip * nXc;
#pragma unroll
                        for (int m = 0; m < nXc; ++m) o[m] += sacc[m];
                    }
                } else {
                    const int ntx = lX + 1;                          // EX[i*ntx + t]: E^t_i of the one-centre expansion
                    for (int i = lane; i < nhb * nXc; i += 32) {
                        const int ip = i / nXc, c = i - ip * nXc;
                        const uint32_t wp = s_herm[ip];
                        int ex, ey, ez;
                        unpack_tuv(cx[c], ex, ey, ez);
                        double s = 0.0;
                        constexpr int st = TWO ? 1 : 2;              // Eq. 12 (one centre): E^t_i = 0 unless t = i mod 2
                        const double *EY = TWO ? EX + ntx * ntx : EX, *EZ = TWO ? EX + 2 * ntx * ntx : EX;
                        for (int t2 = TWO ? 0 : ex & 1; t2 <= ex; t2 += st)
                            for (int u2 = TWO ? 0 : ey & 1; u2 <= ey; u2 += st)
                                for (int v2 = TWO ? 0 : ez & 1; v2 <= ez; v2 += st) {
                                    const double e3 = EX[ex * ntx + t2] * EY[ey * ntx + u2] * EZ[ez * ntx + v2];
                                    const uint32_t wq = (uint32_t)t2 | (uint32_t)u2 << 8 | (uint32_t)v2 << 16 | (uint32_t)(t2 + u2 + v2) << 24;
                                    const double r = R0[hl_herm_index(wp + wq)];
                                    s = ((t2 + u2 + v2) & 1) ? fma(-e3, r, s) : fma(e3, r, s);
                                }
                        G[i] += s;
                    }
                }
            }
            __syncwarp();
            // acc[a b][c] += sum over the box t <= ax+bx, u <= ay+by, v <= az+bz of E^t E^u E^v G[tuv][c]; 7 columns at a time.
            // (A tensor-core form of this step, rows = pairs, K = p~, was measured 1.4x SLOWER: its K loop is one dependent
            // load chain per step and the padded G / acc slices halve the resident warps; profiles/r02_eri3s.md.)
            const double *Ex = E, *Ey = E + esz, *Ez = E + 2 * esz;
            for (int ab = lane; ab < nab_c; ab += 32) {
                const int a = ab / ncb, b = ab - a * ncb;
                int ax, ay, az, bx, by, bz;
                unpack_tuv(ca[a], ax, ay, az);
                unpack_tuv(cb[b], bx, by, bz);
                const double *ex = Ex + (ax * (lb + 1) + bx) * nt, *ey = Ey + (ay * (lb + 1) + by) * nt, *ez = Ez + (az * (lb + 1) + bz) * nt;
#pragma unroll
                for (int c0 = 0; c0 < nXc; c0 += CW) {
                    double r[CW];
#pragma unroll
                    for (int c = 0; c < CW; ++c) r[c] = 0.0;
                    // ONE flat loop over the lane's own box with per-lane counters: nested loops with lane-dependent bounds would
                    // make the warp walk the union of all boxes (84 steps for (ff|) instead of the largest one (27)
                    const int nx = ax + bx, ny = ay + by, nz = az + bz, box = (nx + 1) * (ny + 1) * (nz + 1);
                    int tt = 0, uu = 0, vv = 0;
                    for (int i = 0; i < box; ++i) {
                        const double e3 = ex[tt] * ey[uu] * ez[vv];
                        const double *row = G + cube[(tt * nt + uu) * nt + vv] * nXc + c0;
#pragma unroll
                        for (int c = 0; c < CW; ++c)
                            if (c0 + c < nXc) r[c] = fma(e3, row[c], r[c]);
                        if (++vv > nz) { vv = 0; if (++uu > ny) { uu = 0; ++tt; } }
                    }
                    double *o = acc + ab * nXc + c0;
#pragma unroll
                    for (int c = 0; c < CW; ++c)
                        if (c0 + c < nXc) o[c] += r[c];
                }
            }
        }
        __syncwarp();
        double *out = g.out + t * g.s_t;
        if (!PURE && !(TWO && g.pure)) {
            for (int i = lane; i < nab_c * nXc; i += 32) { const int ab = i / nXc, c = i - ab * nXc; out[ab * g.s_ab + c * g.s_c] = acc[i]; }
        } else {
            // Eq. 16 on a, then on b, through the R / G region (free now)
            const int nsa = nsolid(la), nsb = nsolid(lb);
            double *T1 = W;                                          // [ma][b][c]
            const int nbc = ncb * nXc;
            for (int bc = lane; bc < nbc; bc += 32) {                // lane = (b, c): 7 accumulators over ma, C^{la}[a][ma] broadcast
                double tacc[7];
#pragma unroll
                for (int m = 0; m < 7; ++m) tacc[m] = 0.0;
                for (int a = 0; a < nca; ++a) {
                    const double v = acc[a * nbc + bc];
                    const double *c = CaT + a * MD_HL_CSTR;
#pragma unroll
                    for (int m = 0; m < 7; ++m)
                        if (m < nsa) tacc[m] = fma(c[m], v, tacc[m]);
                }
#pragma unroll
                for (int m = 0; m < 7; ++m)
                    if (m < nsa) T1[m * nbc + bc] = tacc[m];
            }
            __syncwarp();
            for (int i = lane; i < nsa * nXc; i += 32) {             // lane = (ma, c): 7 accumulators over mb
                const int ma = i / nXc, c = i - ma * nXc;
                double oacc[7];
#pragma unroll
                for (int m = 0; m < 7; ++m) oacc[m] = 0.0;
                for (int b = 0; b < ncb; ++b) {
                    const double v = T1[(ma * ncb + b) * nXc + c];
                    const double *cc = CbT + b * MD_HL_CSTR;
#pragma unroll
                    for (int m = 0; m < 7; ++m)
                        if (m < nsb) oacc[m] = fma(cc[m], v, oacc[m]);
                }
                if constexpr (TWO) {                                 // c is still Cartesian: [ma mb][c] goes to the acc region (free now)
#pragma unroll
                    for (int m = 0; m < 7; ++m)
                        if (m < nsb) acc[(ma * nsb + m) * nXc + c] = oacc[m];
                } else {
#pragma unroll
                    for (int m = 0; m < 7; ++m)
                        if (m < nsb) out[(ma * nsb + m) * g.s_ab + c * g.s_c] = oacc[m];
                }
            }
            if constexpr (TWO) {                                     // Eq. 16 on d, then on c
                __syncwarp();
                const int nsx = nsolid(lX), nsd = nsolid(lD), nmab = nsa * nsb;
                double *T2 = W;                                      // [ma mb][c][md] (the R / G region again)
                for (int i = lane; i < nmab * ncx * nsd; i += 32) {
                    const int md = i % nsd, r2 = i / nsd;            // r2 = mab ncx + c
                    double v = 0.0;
                    for (int d = 0; d < ncdd; ++d) v = fma(CdT[d * MD_HL_CSTR + md], acc[r2 * ncdd + d], v);
                    T2[i] = v;
                }
                __syncwarp();
                for (int i = lane; i < nmab * nsx * nsd; i += 32) {
                    const int md = i % nsd, r2 = i / nsd, mc = r2 % nsx, ab = r2 / nsx;
                    double v = 0.0;
                    for (int c = 0; c < ncx; ++c) v = fma(CxT[c * MD_HL_CSTR + mc], T2[(ab * ncx + c) * nsd + md], v);
                    out[ab * g.s_ab + (mc * nsd + md) * g.s_c] = v;
                }
            }
        }
        __syncwarp();
    }
}

}  // namespace mdb
