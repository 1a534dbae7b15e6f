// mma.cuh -- runtime-l quartet kernel whose two Hermite->AO contractions (Eqs. 25-26)
// run as FP64 tensor-core products (mma.sync.m8n8k4.f64, SASS DMMA).  tcgen05 has no FP64
// kind, so mma.sync is the only tensor path this workload has on sm_100a.
//
// Per quartet the CTA (8 warps) evaluates
//   GEMM1  [p~|cd] = sum_kk sum_q~  [p~+q~]^(0)(kb,kk) * Hk(kk)[q~][cd]        (Eqs. 19, 25)
//            M = stacked rows (kb, p~), N = a tile of cd, K = q~; the A operand is never
//            materialised: each lane GATHERS its element [p~+q~]^(0) from the compact
//            Hermite Coulomb tensor in shared memory (Hankel structure of Eq. 19);
//   GEMM2  [ab|cd] += sum_(kb,p~) Hb(kb)[p~][ab] * [p~|cd]                      (Eq. 26)
//            M = ab, N = the cd tile, K = the stacked rows; [p~|cd] goes through shared memory.
// Hb / Hk are the dense Hermite->AO matrices of pair_setup_kernel (Eq. 17: solid harmonics and
// the ket sign already folded in), read from the workspace through L1/L2.
//
// The Hermite Coulomb tensors (Eqs. 21-24) of a whole batch of primitive quartets are built
// together: one warp per tensor, level by level between two ping-pong buffers, so that a CTA
// barrier is paid once per level for the batch, not once per primitive quartet.
#pragma once
#include "boys.cuh"
#include "common.cuh"

namespace mdb {

// CTA size is a template parameter (4 or 8 warps): small classes run faster with four CTAs of 4 warps per SM,
// the largest ones with two CTAs of 8 warps (measured; the host picks, mma_inst.cu).

struct MmaArgs {
    const double *rec_bra, *rec_ket;     // pair_setup_kernel records
    long long stride_bra, stride_ket;
    int Kbra, Kket;
    int Lb, Lk, nab, ncd;
    int kq0;                             // first ket Hermite row with a non-zero H (one-centre solid kets)
    int rslots;                          // Hermite Coulomb tensors resident in shared memory
    int cached;                          // 1: all Kbra*Kket tensors are built once per quartet
    int blk_nkb, blk_np;                 // row-block: blk_nkb bra primitives x blk_np Hermite rows
    const int32_t *qidx;
    long long nq, nket;
    double *out;
    long long s_q, s_bi, s_ki, s_ab, s_cd;
    const double *boys_tab;
    const uint32_t *rlut;                // [2*N~(24)]: recursion neighbours, packed (t,u,v,n)
};

__device__ __forceinline__ void dmma884(double &c0, double &c1, double a, double b) {
    asm("mma.sync.aligned.m8n8k4.row.col.f64.f64.f64.f64 {%0,%1}, {%2}, {%3}, {%0,%1};"
        : "+d"(c0), "+d"(c1) : "d"(a), "d"(b));
}

// Compact index of the Hermite triple whose packed word (t | u<<8 | v<<16 | n<<24) is w:
//   n(n+1)(n+2)/6 + (n-t)(n-t+1)/2 + v          (degree-sorted list of common.cuh)
// x/6 for x = n(n+1)(n+2) <= 15600 (always a multiple of 6) is (x*10923)>>16.
__device__ __forceinline__ int herm_index_packed(uint32_t w) {
    const int n = w >> 24, t = w & 0xff, v = (w >> 16) & 0xff, a = n - t;
    return ((n * (n + 1) * (n + 2) * 10923) >> 16) + ((a * (a + 1)) >> 1) + v;
}

template <int MW, int NW, int MD_MMA_WARPS>
struct MmaCfg {
    static constexpr int ROWS = 8 * MD_MMA_WARPS * MW;            // stacked rows per row-block
    static constexpr int NT = 8 * NW;               // cd columns per pass
    static constexpr int NTS = NT + 4;              // row stride of [p~|cd]: conflict-free B-fragment loads
};

// Shared-memory carve-up (doubles), shared by host and device.
struct MmaSmem {
    int o_r0, o_r1, o_g0, o_pq, o_hdr, o_half, o_rowinfo, o_rowoff, total;
    int rs0, rs1;
};
__host__ __device__ inline MmaSmem mma_smem_layout(int L, int rslots, int Kbra, int Kket, int rows, int nts) {
    auto even = [](int x) { return x + (x & 1); };
    MmaSmem s;
    s.rs0 = even(nherm(L));
    s.rs1 = even(L > 0 ? nherm(L - 1) : 1);
    s.o_r0 = 0;
    s.o_r1 = s.o_r0 + rslots * s.rs0;
    s.o_g0 = s.o_r1 + rslots * s.rs1;
    s.o_pq = s.o_g0 + even(rslots * (L + 1));
    s.o_hdr = s.o_pq + even(rslots * 3);
    s.o_half = s.o_hdr + 4 * (Kbra + Kket);
    s.o_rowinfo = s.o_half + rows * nts;
    s.o_rowoff = s.o_rowinfo + rows;              // rowinfo: 2 ints per row
    s.total = s.o_rowoff + even(rows) / 2;
    return s;
}

template <int MW, int NW, int MD_MMA_WARPS>
__global__ void __launch_bounds__(32 * MD_MMA_WARPS, 16 / MD_MMA_WARPS) eri_mma_kernel(MmaArgs g) {
    constexpr int MD_MMA_THREADS = 32 * MD_MMA_WARPS;
    using C = MmaCfg<MW, NW, MD_MMA_WARPS>;
    extern __shared__ double sm[];
    const int L = g.Lb + g.Lk;
    const int nhb = nherm(g.Lb), nhk = nherm(g.Lk);
    const MmaSmem lay = mma_smem_layout(L, g.rslots, g.Kbra, g.Kket, C::ROWS, C::NTS);
    double *R0 = sm + lay.o_r0, *R1 = sm + lay.o_r1;           // even / odd recursion levels
    double *G0 = sm + lay.o_g0, *PQ = sm + lay.o_pq, *hdr = sm + lay.o_hdr, *half = sm + lay.o_half;
    int2 *rowinfo = (int2 *)(sm + lay.o_rowinfo);              // .x = packed (t,u,v,n) of p~, .y = tensor slot of kb
    int *rowoff = (int *)(sm + lay.o_rowoff);                  // offset of H row (kb,p~) inside the bra pair's records
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const int lr = lane >> 2, lc = lane & 3;                   // fragment row / column of this lane
    const uint2 *lut = (const uint2 *)g.rlut;

    const int nnt_total = (g.ncd + 7) >> 3;
    const int n_rowblk_p = (nhb + g.blk_np - 1) / g.blk_np;    // > 1 only when blk_nkb == 1
    const int n_rowblk_k = (g.Kbra + g.blk_nkb - 1) / g.blk_nkb;

    // Build the tensors of bra primitives [kb0, kb0+nkb) x ket primitives [kk0, kk0+nkk) into slots
    // (kk-kk0)*nkb + (kb-kb0).  Ends with a barrier.
    auto build_R = [&](int kb0, int nkb, int kk0, int nkk) {
        const int nR = nkb * nkk;
        for (int it = tid; it < nR * (L + 1); it += MD_MMA_THREADS) {
            const int s = it / (L + 1), m = it - s * (L + 1);
            const double *hb = hdr + 4 * (kb0 + s % nkb), *hk = hdr + 4 * (g.Kbra + kk0 + s / nkb);
            const double p = hb[0], q = hk[0];
            const double X = hb[1] - hk[1], Y = hb[2] - hk[2], Z = hb[3] - hk[3];
            const double rho = p * q / (p + q);
            const double T = rho * (X * X + Y * Y + Z * Z);
            double f = 34.98683665524972497 / (p * q * sqrt(p + q)) * boys_single(m, T, g.boys_tab);   // 2 pi^{5/2}
            const double m2r = -2.0 * rho;
            for (int i = 0; i < m; ++i) f *= m2r;
            G0[s * (L + 1) + m] = f;
            if (m == L) ((L & 1) ? R1 + s * lay.rs1 : R0 + s * lay.rs0)[0] = f;
            if (m == 0) { PQ[3 * s] = X; PQ[3 * s + 1] = Y; PQ[3 * s + 2] = Z; }
        }
        __syncthreads();
        for (int m = L - 1; m >= 0; --m) {                     // Eq. 24: level m from level m+1
            const int ne = nherm(L - m);
            for (int s = warp; s < nR; s += MD_MMA_WARPS) {
                const double *old = (m & 1) ? R0 + s * lay.rs0 : R1 + s * lay.rs1;
                double *nw = (m & 1) ? R1 + s * lay.rs1 : R0 + s * lay.rs0;
                const double *pq = PQ + 3 * s;
                for (int e = lane; e < ne; e += 32) {
                    const uint32_t w = __ldg(&lut[e].x);
                    double val;
                    if (e == 0) val = G0[s * (L + 1) + m];
                    else {
                        val = pq[w >> 24 & 3] * old[w & 0xfff];
                        const int cf = w >> 26;
                        if (cf) val = fma((double)cf, old[w >> 12 & 0xfff], val);
                    }
                    nw[e] = val;
                }
            }
            __syncthreads();
        }
    };

    for (long long q = blockIdx.x; q < g.nq; q += gridDim.x) {
        long long bi, ki;
        if (g.qidx) { bi = g.qidx[2 * q]; ki = g.qidx[2 * q + 1]; }
        else { bi = q / g.nket; ki = q % g.nket; }
        double *out = g.out + q * g.s_q + bi * g.s_bi + ki * g.s_ki;
        const double *recb = g.rec_bra + bi * g.Kbra * g.stride_bra;
        const double *reck = g.rec_ket + ki * g.Kket * g.stride_ket;

        __syncthreads();                                       // previous quartet is done with shared memory
        for (int it = tid; it < 4 * (g.Kbra + g.Kket); it += MD_MMA_THREADS) {
            const int k = it >> 2, c = it & 3;
            hdr[it] = k < g.Kbra ? recb[k * g.stride_bra + c] : reck[(k - g.Kbra) * g.stride_ket + c];
        }
        __syncthreads();
        if (g.cached) build_R(0, g.Kbra, 0, g.Kket);

        for (int nt0 = 0; nt0 < nnt_total; nt0 += NW) {        // cd pass: NW column tiles
            const int nnt = min(NW, nnt_total - nt0);
            const int cd0 = nt0 * 8;
            bool first = true;                                 // first contribution to out[:, this pass]
            for (int rbk = 0; rbk < n_rowblk_k; ++rbk)
            for (int rbp = 0; rbp < n_rowblk_p; ++rbp) {
                const int kb0 = rbk * g.blk_nkb, nkb = min(g.blk_nkb, g.Kbra - kb0);
                const int p0 = rbp * g.blk_np, np = min(g.blk_np, nhb - p0);
                const int rows = nkb * np, nmt = (rows + 7) >> 3;
                for (int r = tid; r < nmt * 8; r += MD_MMA_THREADS) {
                    const int rr = min(r, rows - 1), kbl = rr / np, ip = p0 + rr - kbl * np;
                    rowinfo[r] = make_int2((int)__ldg(&lut[ip].y), g.cached ? kb0 + kbl : kbl);
                    rowoff[r] = r < rows ? (int)((kb0 + kbl) * g.stride_bra + 4 + (long long)ip * g.nab) : -1;
                }
                __syncthreads();
                uint32_t wrow[MW];
                int slot[MW];
#pragma unroll
                for (int i = 0; i < MW; ++i) {
                    const int j = i * MD_MMA_WARPS + warp;
                    const int2 ri = rowinfo[min(j, nmt - 1) * 8 + lr];
                    wrow[i] = (uint32_t)ri.x; slot[i] = ri.y;
                }
                double acc[MW][NW][2];
#pragma unroll
                for (int i = 0; i < MW; ++i)
#pragma unroll
                    for (int n = 0; n < NW; ++n) acc[i][n][0] = acc[i][n][1] = 0.0;

                const int nslot_kb = g.cached ? g.Kbra : nkb;
                const int kkb = g.cached ? g.Kket : max(1, g.rslots / nkb);   // ket primitives per tensor batch
                for (int kk0 = 0; kk0 < g.Kket; kk0 += kkb) {
                    const int nkk = min(kkb, g.Kket - kk0);
                    if (!g.cached) build_R(kb0, nkb, kk0, nkk);
                    for (int kk = kk0; kk < kk0 + nkk; ++kk) {
                        const double *Hk = reck + kk * g.stride_ket + 4;
                        const double *Rk = R0 + (g.cached ? kk : kk - kk0) * nslot_kb * lay.rs0;
                        const int col = cd0 + lr;
#pragma unroll 2
                        for (int k0 = g.kq0; k0 < nhk; k0 += 4) {
                            const int kq = k0 + lc;
                            const bool kin = kq < nhk;
                            const uint32_t wq = __ldg(&lut[kin ? kq : 0].y);
                            double bfr[NW];
#pragma unroll
                            for (int n = 0; n < NW; ++n)
                                bfr[n] = (kin && n < nnt && col + 8 * n < g.ncd) ? __ldg(Hk + (long long)kq * g.ncd + col + 8 * n) : 0.0;
#pragma unroll
                            for (int i = 0; i < MW; ++i) {
                                if (i * MD_MMA_WARPS + warp < nmt) {
                                    const double a = Rk[slot[i] * lay.rs0 + herm_index_packed(wrow[i] + wq)];
#pragma unroll
                                    for (int n = 0; n < NW; ++n)
                                        if (n < nnt) dmma884(acc[i][n][0], acc[i][n][1], a, bfr[n]);
                                }
                            }
                        }
                    }
                    if (!g.cached) __syncthreads();            // before the next batch overwrites the tensors
                }
                // [p~|cd] -> shared memory
#pragma unroll
                for (int i = 0; i < MW; ++i) {
                    const int j = i * MD_MMA_WARPS + warp;
                    if (j < nmt) {
#pragma unroll
                        for (int n = 0; n < NW; ++n)
                            if (n < nnt)
                                *(double2 *)(half + (j * 8 + lr) * C::NTS + n * 8 + 2 * lc) = make_double2(acc[i][n][0], acc[i][n][1]);
                    }
                }
                __syncthreads();
                // GEMM2: a warp owns ab tiles (round-robin) and, for each, all cd tiles of the pass: one A fragment of
                // Hb (global memory) feeds up to NW DMMAs, the B fragments come from [p~|cd] in shared memory.
                const int nmt2 = (g.nab + 7) >> 3;
                const int ksteps = (rows + 3) >> 2;
                if (nmt2 >= 2 * MD_MMA_WARPS)
                for (int um = warp; um < nmt2; um += MD_MMA_WARPS) {
                    double c2[NW][2];
#pragma unroll
                    for (int n = 0; n < NW; ++n) c2[n][0] = c2[n][1] = 0.0;
                    const int ab = um * 8 + lr;
                    const bool abin = ab < g.nab;
#pragma unroll 2
                    for (int ks = 0; ks < ksteps; ++ks) {
                        const int r = ks * 4 + lc;
                        const int ro = rowoff[r];
                        const double afr = (ro >= 0 && abin) ? __ldg(recb + ro + ab) : 0.0;
                        const double *hrow = half + r * C::NTS + lr;
#pragma unroll
                        for (int n = 0; n < NW; ++n)
                            if (n < nnt) dmma884(c2[n][0], c2[n][1], afr, hrow[n * 8]);
                    }
                    if (abin) {
#pragma unroll
                        for (int n = 0; n < NW; ++n) {
                            if (n >= nnt) continue;
                            const int cd = cd0 + n * 8 + 2 * lc;
                            double *o = out + ab * g.s_ab + cd * g.s_cd;
                            if (cd < g.ncd) { if (first) *o = c2[n][0]; else *o += c2[n][0]; }
                            if (cd + 1 < g.ncd) { if (first) o[g.s_cd] = c2[n][1]; else o[g.s_cd] += c2[n][1]; }
                        }
                    }
                }
                else {
                // few ab tiles: units (ab tile, cd tile) round-robin over the warps, U2 units per warp per chunk
                constexpr int U2 = 4;
                const int nunits = nmt2 * nnt;
                for (int u0 = 0; u0 < nunits; u0 += U2 * MD_MMA_WARPS) {
                    double c2[U2][2];
                    int um[U2], un[U2];
#pragma unroll
                    for (int i = 0; i < U2; ++i) {
                        c2[i][0] = c2[i][1] = 0.0;
                        const int u = u0 + i * MD_MMA_WARPS + warp;
                        um[i] = u < nunits ? u / nnt : -1;
                        un[i] = u < nunits ? u - um[i] * nnt : 0;
                    }
#pragma unroll 2
                    for (int ks = 0; ks < ksteps; ++ks) {
                        const int r = ks * 4 + lc;
                        const int ro = rowoff[r];
                        double afr[U2], bfr2[U2];
#pragma unroll
                        for (int i = 0; i < U2; ++i) {
                            const int ab = um[i] * 8 + lr;
                            afr[i] = (um[i] >= 0 && ro >= 0 && ab < g.nab) ? __ldg(recb + ro + ab) : 0.0;
                            bfr2[i] = half[r * C::NTS + un[i] * 8 + lr];
                        }
#pragma unroll
                        for (int i = 0; i < U2; ++i)
                            if (um[i] >= 0) dmma884(c2[i][0], c2[i][1], afr[i], bfr2[i]);
                    }
#pragma unroll
                    for (int i = 0; i < U2; ++i) {
                        if (um[i] < 0) continue;
                        const int ab = um[i] * 8 + lr, cd = cd0 + un[i] * 8 + 2 * lc;
                        if (ab >= g.nab) continue;
                        double *o = out + ab * g.s_ab + cd * g.s_cd;
                        if (cd < g.ncd) { if (first) *o = c2[i][0]; else *o += c2[i][0]; }
                        if (cd + 1 < g.ncd) { if (first) o[g.s_cd] = c2[i][1]; else o[g.s_cd] += c2[i][1]; }
                    }
                }
                }
                first = false;
                __syncthreads();                               // half / rowinfo are rewritten by the next row-block
            }
        }
    }
}

}  // namespace mdb
