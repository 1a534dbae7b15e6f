// hl.cuh -- the high-l quartet kernel: steps S1-S5 in ONE launch for classes with an l >= 3 shell.
//
// One persistent CTA evaluates one quartet (or triplet) at a time:
//   S1  per primitive pair of both sides: the three 1-D Hermite tables (Eqs. 9, 10, 13, 14) by a warp
//       per Cartesian axis, then the dense Hermite->AO matrices H (Eq. 17: solid harmonics folded in, ket sign
//       of Eq. 19 folded in) by all threads, register-blocked, one index at a time.  The matrices go to a
//       PER-CTA scratch in global memory (L2), never to a per-pair workspace: the scratch of the whole grid is a
//       few hundred MB whatever the number of quartets (no N_shells^2 data is stored);
//   S2-S3  Boys function and the Hermite Coulomb tensors [r~]^(0) of all primitive quartets, level by level
//       (Eqs. 21-24), in shared memory;
//   S4  per cd tile of NT = 8 NW columns, both contractions on the FP64 tensor path (mma.sync.m8n8k4.f64):
//         GEMM1  [p~|cd] = sum_kk sum_q~ [p~+q~]^(0) Hk(kk)[q~][cd]   (Eqs. 19, 25), A gathered from the tensor,
//         GEMM2  [ab|cd] = sum_(kb,p~) Hb(kb)[p~][ab] [p~|cd]          (Eq. 26),
//       with BOTH H operands streamed from the scratch into a shared-memory ring by cp.async.bulk (TMA bulk
//       copies) completing on mbarriers, a few chunks ahead of the tensor-core loop;
//   S5  the accumulators of GEMM2 are the final [ab|cd] tile: stored once, no read-modify-write.
// tcgen05 has no FP64 kind, so mma.sync is the only tensor path FP64 has on sm_100a.
#pragma once
#include <type_traits>

#include "boys.cuh"
#include "common.cuh"

namespace mdb {

#define MD_HL_KC1 32          // ket Hermite rows per ring chunk of GEMM1
#define MD_HL_STAGES 4
#define MD_HL_MT2 3           // ab row tiles per warp in GEMM2 (register-resident output)
#define MD_HL_CSTR 16         // row stride of the transposed Cartesian->solid tables [cart][m], zero-padded

struct HlArgs {
    PairView bra, ket;
    int pure;
    int la, lb, lc, ld;                  // ld = 0 for a one-centre ket
    int Ka, Kb, Kc, Kd, Kbra, Kket;
    int Lb, Lk, nab, ncd, nhb, nhk;
    int kbb, nblk;                       // bra primitives per row block of [p~|cd] (what fits shared memory); blocks
    int mrows, mrows_pad;                // stacked rows (kb, p~) of one row block (kbb*nhb); padded to a multiple of kc2
    int kc2;                             // stacked bra rows per ring chunk of GEMM2: 8 or 16
    int nhk_pad;                         // ket Hermite rows padded to MD_HL_KC1
    int sb;                              // row stride of Hb in the scratch: >= 8*ceil(nab/8), = 4 mod 16
    int ntile;                           // cd tiles
    int q_first;                         // first GEMM1 chunk row with a non-zero Hk (one-centre solid kets), multiple of KC1
    double *scratch;                     // fused mode: [grid][scratch_stride]
    int fused;                           // 1: S1 runs inside the quartet kernel into the CTA's scratch; 0: pair records
    int by_quartet;                      // record mode: 1 = record r belongs to quartet q_begin + r, 0 = to pair r
    int qswap;                           // 1: the kernel's bra is the CALLER's ket (index columns and product order swapped)
    const double *rec_b, *rec_k;         // record mode: H records of hl_pair_kernel (same layout as the scratch halves)
    const double *hdr_b, *hdr_k;         // record mode: {p, Px, Py, Pz} per record and primitive
    long long rec_stride_b, rec_stride_k;
    long long q_begin, q_end;            // quartets of this launch
    long long scratch_stride, off_hk;    // doubles per CTA; offset of the ket part
    const int32_t *qidx;
    long long nq, nket;
    double *out;
    long long s_q, s_bi, s_ki, s_ab, s_cd;
    const double *boys_tab;
    const uint32_t *rlut;
    // shared-memory carve-up (doubles from the base)
    int o_herm, o_rowinfo, o_ct, o_hdr, o_bar, o_r0, o_g0, o_pq, o_ov, o_ring, total;
    int rs0, rs1, ov_doubles, ring_stage;
};

// ---- mbarrier / bulk-copy primitives (PTX ISA: mbarrier, cp.async.bulk) -------------------------------------------
__device__ __forceinline__ uint32_t hl_saddr(const void *p) { return (uint32_t)__cvta_generic_to_shared(p); }
__device__ __forceinline__ void hl_bar_init(uint64_t *b, int count) {
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(hl_saddr(b)), "r"(count));
}
__device__ __forceinline__ void hl_bar_expect(uint64_t *b, uint32_t bytes) {
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(hl_saddr(b)), "r"(bytes) : "memory");
}
__device__ __forceinline__ void hl_bar_arrive(uint64_t *b) {
    asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];" ::"r"(hl_saddr(b)) : "memory");
}
__device__ __forceinline__ void hl_bar_wait(uint64_t *b, uint32_t parity) {
    asm volatile(
        "{\n .reg .pred p;\n WAIT_%=:\n mbarrier.try_wait.parity.shared::cta.b64 p, [%0], %1;\n @p bra DONE_%=;\n bra WAIT_%=;\n DONE_%=:\n}"
        ::"r"(hl_saddr(b)), "r"(parity) : "memory");
}
__device__ __forceinline__ void hl_bulk_g2s(void *dst, const void *src, uint32_t bytes, uint64_t *b) {
    asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];"
                 ::"r"(hl_saddr(dst)), "l"(src), "r"(bytes), "r"(hl_saddr(b)) : "memory");
}

__device__ __forceinline__ void hl_dmma884(double &c0, double &c1, double a, double b) {
    asm("mma.sync.aligned.m8n8k4.row.col.f64.f64.f64.f64 {%0,%1}, {%2}, {%3}, {%0,%1};"
        : "+d"(c0), "+d"(c1) : "d"(a), "d"(b));
}

// Compact index of the Hermite triple with packed word w = t | u<<8 | v<<16 | n<<24 (degree-sorted list, common.cuh).
__device__ __forceinline__ int hl_herm_index(uint32_t w) {
    const int n = w >> 24, t = w & 0xff, v = (w >> 16) & 0xff, a = n - t;
    return ((n * (n + 1) * (n + 2) * 10923) >> 16) + ((a * (a + 1)) >> 1) + v;
}

// hl_e_axis_warp (one Cartesian axis of the two-centre Hermite expansion by one warp) lives in common.cuh: pair.cuh uses it too.

// Where H[p~][m] of one primitive pair goes in the CTA's scratch.
struct HlBraDst {            // [kb*nhb + p~][sb]
    double *base; int sb;
    __device__ __forceinline__ double *operator()(int p, int m) const { return base + (long long)p * sb + m; }
    __device__ __forceinline__ long long row(int p) const { return (long long)p * sb; }
    __device__ __forceinline__ int col(int m) const { return m; }
};
template <int NT>
struct HlKetDst {            // tile-major: [cd tile][kk][q~ (padded)][NT + 4]
    double *base; long long tile_stride;     // Kket * nhk_pad * (NT+4)
    __device__ __forceinline__ double *operator()(int q, int m) const {
        const int j = m / NT, n = m - j * NT;
        return base + j * tile_stride + (long long)q * (NT + 4) + n;
    }
    __device__ __forceinline__ long long row(int q) const { return (long long)q * (NT + 4); }
    __device__ __forceinline__ int col(int m) const { const int j = m / NT; return (int)(j * tile_stride) + m - j * NT; }
};

// ---- S1: dense H of one primitive pair (Eqs. 7, 17), all threads of the CTA ---------------------------------
//   Cartesian: H[p~][ab]   = c E^t_{ax bx} E^u_{ay by} E^v_{az bz}
//   solid    : H[p~][mamb] = c sum_a C^{la}_{ma,a} sum_b C^{lb}_{mb,b} E^{ab}_{p~}, one index at a time:
//     stage A  task (p~, a):  T1[p~][a][mb] = sum_b C^{lb}[mb][b] E^{ab}_{p~}   (13 accumulators in registers)
//     stage B  task (p~, mb): H[p~][ma][mb] = c sum_a C^{la}[ma][a] T1[p~][a][mb]
//   Steps whose operand is zero for the whole warp are skipped (Eq. 14 makes 80 % of E^{ab}_{p~} vanish).
// E = the three axis tables (shared memory), T1 = shared scratch of t1cap doubles, CaT/CbT = transposed
// Cartesian->solid tables [cart][MD_HL_CSTR].  Ends with a barrier.  neg: fold (-1)^{|q~|} (Eq. 19).
template <int NTHR, class Dst>
__device__ __forceinline__ void hl_build_H(int la, int lb, int pure, bool neg, double coef, const double *E, double *T1,
                                           int t1cap, const uint32_t *s_herm, const double *CaT, const double *CbT,
                                           const Dst &dst) {
    const int tid = threadIdx.x;
    const int Lb = la + lb, nt = Lb + 1, nh = nherm(Lb), esz = (la + 1) * (lb + 1) * nt;
    const int nca = ncart(la), ncb = ncart(lb);
    const uint32_t *ca = s_herm + nherm(la - 1), *cb = s_herm + nherm(lb - 1);
    const double *Ex = E, *Ey = E + esz, *Ez = E + 2 * esz;
    if (!pure) {
        const int nab = nca * ncb;
        for (int e = tid; e < nh * nab; e += NTHR) {
            const int ih = e / nab, ab = e - ih * nab, a = ab / ncb, b = ab - a * ncb;
            int t, u, v, ax, ay, az, bx, by, bz;
            unpack_tuv(s_herm[ih], t, u, v);
            unpack_tuv(ca[a], ax, ay, az);
            unpack_tuv(cb[b], bx, by, bz);
            double val = coef * Ex[(ax * (lb + 1) + bx) * nt + t] * Ey[(ay * (lb + 1) + by) * nt + u] *
                         Ez[(az * (lb + 1) + bz) * nt + v];
            if (neg && ((t + u + v) & 1)) val = -val;
            *dst(ih, ab) = val;
        }
        __syncthreads();
        return;
    }
    // Both stages on the FP64 tensor path (mma.sync.m8n8k4.f64), 8 x 8 tiles, K steps of 4:
    //   stage A  rows (p~, a), columns mb, K = b: a lane forms its own A element E^{ab}_{p~} from the three axis tables;
    //            the B fragments C^{lb}[b][mb] are class constants held in registers.  A K step whose 32 elements all
    //            vanish (Eq. 14) is skipped.
    //   stage B  per p~: rows ma, columns mb, K = a: A fragments C^{la}[a][ma] in registers, B fragments from T1.
    const int nsa = nsolid(la), nsb = nsolid(lb);
    const int lane = tid & 31, warp = tid >> 5, lr = lane >> 2, lc = lane & 3;
    constexpr int NWARPS = NTHR / 32, TS = 20;              // T1 row stride: 16 columns + 4 (conflict-free fragments)
    const int ntb = (nsb + 7) >> 3, nta = (nsa + 7) >> 3;   // column tiles of mb, row tiles of ma (1 or 2)
    const int ksb = (ncb + 3) >> 2, ksa = (nca + 3) >> 2;   // K steps over b and over a (<= 7)
    // A warp owns groups of pw consecutive Hermite rows end to end (stage A into its private T1 slice, stage B out of
    // it), so the loop has no CTA barrier: the LDS-bound stage A of one warp overlaps the tensor-core steps of the others.
    const int pw = nca >= 21 ? 1 : nca >= 10 ? 2 : nca >= 6 ? 4 : 8;      // pw * nca rows: a multiple of 8, or nearly
    double *T1w = T1 + (size_t)warp * pw * nca * TS;                       // needs t1cap >= NWARPS * pw * nca * TS (host)
    (void)t1cap;
    double cbf[7][2], caf[7][2];                            // constant fragments: C^{lb}[b][mb], C^{la}[a][ma]
    // Lane constants of the two stages, so that the inner loops are loads and tensor-core steps only: table offsets of
    // b = 4k + lc on the three axes (b past the shell reads entry 0: finite, and its C^{lb} row is zero), T1 row offsets of
    // a = 4k + lc, and the scratch offsets of the eight H elements this lane owns in stage B.
    int ox[7], oy[7], oz[7], ta[7];
#pragma unroll
    for (int k = 0; k < 7; ++k) {
        const int b = 4 * k + lc;
        int bx = 0, by = 0, bz = 0;
        if (b < ncb) unpack_tuv(cb[b], bx, by, bz);
        ox[k] = bx * nt; oy[k] = by * nt; oz[k] = bz * nt;
        ta[k] = min(b, nca - 1) * TS;                          // a past the shell: any finite row, its C^{la} row is zero
#pragma unroll
        for (int n = 0; n < 2; ++n) {
            cbf[k][n] = b < ncb ? CbT[b * MD_HL_CSTR + 8 * n + lr] : 0.0;
            caf[k][n] = b < nca ? CaT[b * MD_HL_CSTR + 8 * n + lr] : 0.0;    // same lane pattern: a = 4k + lc, ma = 8n + lr
        }
    }
    int hoff[2][2][2];
    bool hval[2][2][2];
#pragma unroll
    for (int i = 0; i < 2; ++i)
#pragma unroll
        for (int n = 0; n < 2; ++n)
#pragma unroll
            for (int e = 0; e < 2; ++e) {
                const int ma = 8 * i + lr, mb = 8 * n + 2 * lc + e;
                hval[i][n][e] = ma < nsa && mb < nsb;
                hoff[i][n][e] = hval[i][n][e] ? dst.col(ma * nsb + mb) : 0;
            }
    for (int h0 = warp * pw; h0 < nh; h0 += NWARPS * pw) {
        const int hc = min(pw, nh - h0);
        const int nrows = hc * nca, nmt = (nrows + 7) >> 3;
        for (int mt = 0; mt < nmt; ++mt) {
            const int r = mt * 8 + lr;
            const bool rv = r < nrows;
            const int rr = rv ? r : nrows - 1;
            const int ih = rr / nca, a = rr - ih * nca;
            int t, u, v, ax, ay, az;
            unpack_tuv(s_herm[h0 + ih], t, u, v);
            unpack_tuv(ca[a], ax, ay, az);
            const double *ex = Ex + ax * (lb + 1) * nt + t, *ey = Ey + ay * (lb + 1) * nt + u, *ez = Ez + az * (lb + 1) * nt + v;
            double c[2][2] = {{0.0, 0.0}, {0.0, 0.0}}, d[2][2] = {{0.0, 0.0}, {0.0, 0.0}};   // even / odd K steps: two chains
            // all operands first (21 loads in flight), then the votes, then the tensor-core steps
            double x[7];
            uint32_t live = 0;
#pragma unroll
            for (int k = 0; k < 7; ++k) x[k] = ex[ox[k]] * ey[oy[k]] * ez[oz[k]];   // rows past the end repeat the last row: not stored
#pragma unroll
            for (int k = 0; k < 7; ++k) live |= (__any_sync(0xffffffffu, x[k] != 0.0) ? 1u : 0u) << k;
#pragma unroll
            for (int k = 0; k < 7; ++k) {
                if (live >> k & 1) {
                    if (k & 1) {
                        hl_dmma884(d[0][0], d[0][1], x[k], cbf[k][0]);
                        if (ntb > 1) hl_dmma884(d[1][0], d[1][1], x[k], cbf[k][1]);
                    } else {
                        hl_dmma884(c[0][0], c[0][1], x[k], cbf[k][0]);
                        if (ntb > 1) hl_dmma884(c[1][0], c[1][1], x[k], cbf[k][1]);
                    }
                }
            }
            c[0][0] += d[0][0]; c[0][1] += d[0][1]; c[1][0] += d[1][0]; c[1][1] += d[1][1];
            double *o = T1w + (size_t)r * TS + 2 * lc;
            if (rv) {
                *(double2 *)o = make_double2(c[0][0], c[0][1]);
                if (ntb > 1) *(double2 *)(o + 8) = make_double2(c[1][0], c[1][1]);
            }
        }
        __syncwarp();
        for (int ih = 0; ih < hc; ++ih) {
            const double *t1 = T1w + (size_t)ih * nca * TS + lr;
            double c[2][2][2] = {{{0.0, 0.0}, {0.0, 0.0}}, {{0.0, 0.0}, {0.0, 0.0}}};      // [ma tile][mb tile][2]
            double b0[7], b1[7];
            uint32_t live = 0;
#pragma unroll
            for (int k = 0; k < 7; ++k) { b0[k] = t1[ta[k]]; b1[k] = ntb > 1 ? t1[ta[k] + 8] : 0.0; }
#pragma unroll
            for (int k = 0; k < 7; ++k) live |= (__any_sync(0xffffffffu, b0[k] != 0.0 || b1[k] != 0.0) ? 1u : 0u) << k;
#pragma unroll
            for (int k = 0; k < 7; ++k) {
                if (live >> k & 1) {
                    hl_dmma884(c[0][0][0], c[0][0][1], caf[k][0], b0[k]);
                    if (ntb > 1) hl_dmma884(c[0][1][0], c[0][1][1], caf[k][0], b1[k]);
                    if (nta > 1) {
                        hl_dmma884(c[1][0][0], c[1][0][1], caf[k][1], b0[k]);
                        if (ntb > 1) hl_dmma884(c[1][1][0], c[1][1][1], caf[k][1], b1[k]);
                    }
                }
            }
            const double sgn = (neg && (s_herm[h0 + ih] >> 24 & 1)) ? -coef : coef;
            double *hrow = dst.base + dst.row(h0 + ih);
#pragma unroll
            for (int i = 0; i < 2; ++i)
#pragma unroll
                for (int n = 0; n < 2; ++n)
#pragma unroll
                    for (int e = 0; e < 2; ++e)
                        if (hval[i][n][e]) hrow[hoff[i][n][e]] = sgn * c[i][n][e];
        }
        __syncwarp();                                       // the slice is rewritten by the warp's next group
    }
    __syncthreads();
}

// One K step (4 ket Hermite rows) of GEMM1 for a warp's MW x NW tiles: the A elements [p~+q~]^(0) are gathered from
// the tensor, the B fragments come from the ring.  FULLN: all NW column tiles of the cd tile exist (no guards, so the
// compiler can overlap the index arithmetic of one step with the tensor-core instructions of the previous one).
template <int MW, int NW, bool FULLN>
__device__ __forceinline__ void hl_gemm1_step(double (&acc)[MW][NW][2], const double *B, const double *Rk,
                                              const int (&rbase)[MW], const uint32_t (&wrow)[MW], uint32_t wq, int nnt) {
    double bfr[NW], a[MW];
#pragma unroll
    for (int n = 0; n < NW; ++n) bfr[n] = B[n * 8];
#pragma unroll
    for (int i = 0; i < MW; ++i) a[i] = Rk[rbase[i] + hl_herm_index(wrow[i] + wq)];
#pragma unroll
    for (int i = 0; i < MW; ++i)
#pragma unroll
        for (int n = 0; n < NW; ++n)
            if (FULLN || n < nnt) hl_dmma884(acc[i][n][0], acc[i][n][1], a[i], bfr[n]);
}

// ---- S1 for one side of one quartet (or one shell pair): every primitive pair's Hermite tables (three warps, one
// per axis), {p, P} header and dense H record.  ws = shared scratch of cap doubles.  rec: bra [K][nh][sb], ket
// [cd tile][K][nh_pad][NT+4] (tile_stride = K nh_pad (NT+4)); bra primitives are grouped kbb to a row block of blk_rows
// rows.  Ends with a barrier.
template <int NTHR, int NT>
__device__ __forceinline__ void hl_side(const PairView &pv, bool ket, int l1, int l2, int K1, int K2, int pure, long long ip,
                                        double *hdr, double *ws, int cap, const uint32_t *s_herm, const double *CaT,
                                        const double *CbT, double *rec, int nh, int nh_pad, int sb, long long tile_stride,
                                        int kbb, int blk_rows) {
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    long long i1 = ip, i2 = ip;
    if (pv.idx) { i1 = pv.idx[2 * ip]; i2 = pv.idx[2 * ip + 1]; }
    const int esz = (l1 + 1) * (l2 + 1) * (l1 + l2 + 1);
    double *E = ws, *T1 = ws + ((3 * esz + 1) & ~1);               // 16-byte aligned rows for the fragment stores
    const int t1cap = cap - ((3 * esz + 1) & ~1);
    for (int kp = 0; kp < K1 * K2; ++kp) {
        const int k1 = kp / K2, k2 = kp - k1 * K2;
        const double za = pv.a.exps[i1 * K1 + k1];
        const double zb = pv.single ? 0.0 : pv.b.exps[i2 * K2 + k2];
        const double coef = pv.a.coefs[i1 * K1 + k1] * (pv.single ? 1.0 : pv.b.coefs[i2 * K2 + k2]);
        if (warp < 3) {
            const double A = pv.a.center[3 * i1 + warp], B = pv.single ? A : pv.b.center[3 * i2 + warp];
            hl_e_axis_warp(l1, l2, za, zb, A - B, E + warp * esz, lane);
            if (lane == 0) {
                double *h = hdr + 4 * kp;
                h[1 + warp] = (za * A + zb * B) / (za + zb);
                if (warp == 0) h[0] = za + zb;
            }
        }
        __syncthreads();
        if (pv.single && pure) {
            // One-centre solid harmonics (Hobson): S_lm(d/dA) e^{-z r_A^2} = (2z)^l S_lm(r_A) e^{-z r_A^2}: only the
            // Hermites of order exactly l appear, with coefficient C^l_{m,q~}/(2z)^l; lower rows are exact zeros.
            const int ns = nsolid(l1), nlow = nherm(l1 - 1);
            double f = coef;
            for (int i = 0; i < l1; ++i) f *= 0.5 / za;
            if (l1 & 1) f = -f;
            HlKetDst<NT> dst{rec + (long long)kp * nh_pad * (NT + 4), tile_stride};
            for (int e = tid; e < nh * ns; e += NTHR) {
                const int ih = e / ns, m = e - ih * ns;
                *dst(ih, m) = ih < nlow ? 0.0 : f * CaT[(ih - nlow) * MD_HL_CSTR + m];
            }
            __syncthreads();
        } else if (ket) {
            HlKetDst<NT> dst{rec + (long long)kp * nh_pad * (NT + 4), tile_stride};
            hl_build_H<NTHR>(l1, l2, pure, true, coef, E, T1, t1cap, s_herm, CaT, CbT, dst);
        } else {
            HlBraDst dst{rec + ((long long)(kp / kbb) * blk_rows + (long long)(kp % kbb) * nh) * sb, sb};   // row block, then primitive
            hl_build_H<NTHR>(l1, l2, pure, false, coef, E, T1, t1cap, s_herm, CaT, CbT, dst);
        }
    }
}

// Constant tables of a CTA: Hermite triples and the transposed, zero-padded Cartesian->solid tables of up to 4 shells.
template <int NTHR>
__device__ __forceinline__ void hl_stage_tables(uint32_t *s_herm, int nhm, double *CT, const int (&ls)[4]) {
    const int tid = threadIdx.x, CTS = 28 * MD_HL_CSTR;
    for (int i = tid; i < nhm; i += NTHR) s_herm[i] = c_herm[i];
    for (int i = tid; i < 4 * CTS; i += NTHR) CT[i] = 0.0;
    __syncthreads();
    for (int s = 0; s < 4; ++s) {
        const int l = ls[s], nc = ncart(l), ns = nsolid(l);
        for (int i = tid; i < nc * ns; i += NTHR) {
            const int m = i / nc, c = i - m * nc;
            CT[s * CTS + c * MD_HL_CSTR + m] = c_solid[solid_off(l) + i];
        }
    }
}

// ---- S1 as a kernel of its own: one H record per CTA iteration (per shell pair, or per quartet side), for the record
// mode of hl_kernel.  Persistent 4-warp CTAs, several per SM.
struct HlPairArgs {
    PairView pv;
    int ket, l1, l2, K1, K2, pure;
    int nh, nh_pad, sb, kbb, blk_rows;
    long long tile_stride;
    long long nrec, rec_stride;
    double *rec, *hdr;                   // [nrec][rec_stride], [nrec][K1*K2][4]
    int by_quartet;                      // record r <- side of quartet q_begin + r instead of pair r
    int qswap;
    const int32_t *qidx;
    long long q_begin, nket;
    int o_herm, o_ct, o_ws, ws_doubles;  // shared-memory carve-up (doubles)
};

template <int NW>
__global__ void __launch_bounds__(128, 4) hl_pair_kernel(HlPairArgs g) {
    constexpr int NTHR = 128, NT = 8 * NW;
    extern __shared__ double sm[];
    uint32_t *s_herm = (uint32_t *)(sm + g.o_herm);
    double *CT = sm + g.o_ct;
    const int ls[4] = {g.l1, g.l2, 0, 0};
    hl_stage_tables<NTHR>(s_herm, nherm(g.l1 + g.l2), CT, ls);
    __syncthreads();
    for (long long r = blockIdx.x; r < g.nrec; r += gridDim.x) {
        long long ip = r;
        if (g.by_quartet) {
            const long long q = g.q_begin + r;
            const int col = g.ket ^ g.qswap;                     // column of the caller's index list / product
            if (g.qidx) ip = g.qidx[2 * q + col];
            else ip = col ? q % g.nket : q / g.nket;
        }
        hl_side<NTHR, NT>(g.pv, g.ket != 0, g.l1, g.l2, g.K1, g.K2, g.pure, ip, g.hdr + r * 4 * g.K1 * g.K2, sm + g.o_ws,
                          g.ws_doubles, s_herm, CT, CT + 28 * MD_HL_CSTR, g.rec + r * g.rec_stride, g.nh, g.nh_pad, g.sb,
                          g.tile_stride, g.kbb, g.blk_rows);
    }
}

// Order in which one quartet's H chunks pass through the ring: for every cd tile, for every row pass of GEMM1 the
// chunks (kk, c) of Hk, then the chunks of Hb for GEMM2; with several bra-primitive row blocks, that per block.  Only the producer thread advances it.
struct HlStream {
    int j, blk, pass, kk, c, c2;
    __device__ __forceinline__ void reset(int c_first) { j = 0; blk = 0; pass = 0; kk = 0; c = c_first; c2 = -1; }
};

template <int MW, int NW, int NWARPS>
__global__ void __launch_bounds__(32 * NWARPS, (NWARPS == 4 ? 3 : 1)) hl_kernel(HlArgs g) {
    constexpr int NTHR = 32 * NWARPS, NT = 8 * NW, NTS = NT + 4, ST = MD_HL_STAGES;
    extern __shared__ double sm[];
    uint32_t *s_herm = (uint32_t *)(sm + g.o_herm);
    int2 *rowinfo = (int2 *)(sm + g.o_rowinfo);            // .x = packed (t,u,v,n) of p~, .y = kb
    double *CT = sm + g.o_ct;                              // 4 transposed Cartesian->solid tables
    double *hdr = sm + g.o_hdr;                            // {p, Px, Py, Pz} per bra primitive, then per ket primitive
    uint64_t *full = (uint64_t *)(sm + g.o_bar), *empty = full + ST;
    double *R0 = sm + g.o_r0, *G0 = sm + g.o_g0, *PQ = sm + g.o_pq;
    double *ov = sm + g.o_ov;                              // [p~|cd] tile; before that R1 / the S1 scratch (spans the ring too)
    double *R1 = ov, *Vp = ov;
    double *ring = sm + g.o_ring;
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const int lr = lane >> 2, lc = lane & 3;
    const int L = g.Lb + g.Lk, nhb = g.nhb, nhk = g.nhk;
    const uint2 *lut = (const uint2 *)g.rlut;
    const int CTS = 28 * MD_HL_CSTR;
    double *scr = g.fused ? g.scratch + (long long)blockIdx.x * g.scratch_stride : nullptr;
    const double *hb = scr, *hk = scr ? scr + g.off_hk : nullptr;   // fused mode; record mode sets them per quartet
    const int nmt = g.mrows_pad >> 3, npass = (nmt + NWARPS * MW - 1) / (NWARPS * MW);
    const int nc1 = g.nhk_pad / MD_HL_KC1, c_first = g.q_first / MD_HL_KC1, nc2 = g.mrows_pad / g.kc2;
    const int nmt2 = (g.nab + 7) >> 3;
    const long long hk_tile = (long long)g.Kket * g.nhk_pad * NTS;
    const uint32_t bytes1 = MD_HL_KC1 * NTS * 8, bytes2 = g.kc2 * g.sb * 8;

    // ---- once per CTA: constant tables, barriers, zeroed scratch (its padding is never written again) ----
    {
        const int ls[4] = {g.la, g.lb, g.lc, g.ld};
        hl_stage_tables<NTHR>(s_herm, nherm(max(g.Lb, g.Lk)), CT, ls);
        for (int r = tid; r < g.mrows_pad; r += NTHR) {            // one row block: .y = bra primitive inside the block
            const int rr = min(r, g.mrows - 1), kb = rr / nhb;
            rowinfo[r] = make_int2((int)c_herm[rr - kb * nhb], kb);
        }
        if (tid == 0) {
            for (int s = 0; s < ST; ++s) { hl_bar_init(full + s, 1); hl_bar_init(empty + s, NWARPS); }
            asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
        }
        if (g.fused) for (long long i = tid; i < g.scratch_stride; i += NTHR) scr[i] = 0.0;
    }
    long long gcons = 0, gprod = 0;                        // chunks consumed (all threads) / issued (thread 0), CTA lifetime
    HlStream ps;
    long long left = 0;                                    // chunks of the current quartet not yet issued (thread 0)
    const long long per_quartet = (long long)g.ntile * g.nblk * ((long long)npass * g.Kket * (nc1 - c_first) + nc2);

    auto produce = [&]() {                                 // thread 0: issue the next chunk of the stream
        const int s = (int)(gprod % ST);
        if (gprod >= ST) hl_bar_wait(empty + s, (uint32_t)((gprod / ST - 1) & 1));
        const double *src;
        uint32_t bytes;
        if (ps.c2 < 0) {
            src = hk + ps.j * hk_tile + ((long long)ps.kk * g.nhk_pad + (long long)ps.c * MD_HL_KC1) * NTS;
            bytes = bytes1;
            if (++ps.c == nc1) { ps.c = c_first; if (++ps.kk == g.Kket) { ps.kk = 0; if (++ps.pass == npass) { ps.pass = 0; ps.c2 = 0; } } }
        } else {
            src = hb + ((long long)ps.blk * g.mrows_pad + (long long)ps.c2 * g.kc2) * g.sb;
            bytes = bytes2;
            if (++ps.c2 == nc2) { ps.c2 = -1; if (++ps.blk == g.nblk) { ps.blk = 0; ++ps.j; } }
        }
        hl_bar_expect(full + s, bytes);
        hl_bulk_g2s(ring + (size_t)s * g.ring_stage, src, bytes, full + s);
        ++gprod; --left;
    };
    auto acquire = [&]() -> const double * {               // all threads: wait for the next chunk
        const int s = (int)(gcons % ST);
        hl_bar_wait(full + s, (uint32_t)((gcons / ST) & 1));
        return ring + (size_t)s * g.ring_stage;
    };
    auto release = [&]() {                                 // all threads: done with it; thread 0 tops the ring up
        __syncwarp();
        if (lane == 0) hl_bar_arrive(empty + (int)(gcons % ST));
        ++gcons;
        if (tid == 0 && left > 0) produce();
    };

    for (long long q = g.q_begin + blockIdx.x; q < g.q_end; q += gridDim.x) {
        long long bi, ki;
        if (g.qidx) { bi = g.qidx[2 * q + g.qswap]; ki = g.qidx[2 * q + 1 - g.qswap]; }
        else if (g.qswap) { bi = q % g.nket; ki = q / g.nket; }     // g.nket = the caller's ket count = this kernel's bra count
        else { bi = q / g.nket; ki = q % g.nket; }
        double *out = g.out + q * g.s_q + bi * g.s_bi + ki * g.s_ki;
        __syncthreads();                                   // the previous quartet is done with shared memory and the scratch

        // ---- S1: Hermite tables and H of every primitive pair of both sides -> scratch (fused mode), or the records ----
        if (g.fused) {
            const int cap = g.ov_doubles + ST * g.ring_stage;
            hl_side<NTHR, NT>(g.bra, false, g.la, g.lb, g.Ka, g.Kb, g.pure, bi, hdr, ov, cap, s_herm, CT, CT + CTS, scr,
                              nhb, 0, g.sb, 0, g.kbb, g.mrows_pad);
            hl_side<NTHR, NT>(g.ket, true, g.lc, g.ld, g.Kc, g.Kd, g.pure, ki, hdr + 4 * g.Kbra, ov, cap, s_herm, CT + 2 * CTS,
                              CT + 3 * CTS, scr + g.off_hk, nhk, g.nhk_pad, 0, hk_tile, 1, 0);
        } else {
            const long long rb = g.by_quartet ? q - g.q_begin : bi, rk = g.by_quartet ? q - g.q_begin : ki;
            hb = g.rec_b + rb * g.rec_stride_b;
            hk = g.rec_k + rk * g.rec_stride_k;
            for (int i = tid; i < 4 * (g.Kbra + g.Kket); i += NTHR)
                hdr[i] = i < 4 * g.Kbra ? g.hdr_b[rb * 4 * g.Kbra + i] : g.hdr_k[rk * 4 * g.Kket + i - 4 * g.Kbra];
        }
        __threadfence();
        asm volatile("fence.proxy.async;" ::: "memory");   // generic-proxy stores to the scratch before the bulk copies read it
        __syncthreads();
        if (tid == 0) {
            ps.reset(c_first);
            left = per_quartet;
            for (int i = 0; i < ST - 1 && left > 0; ++i) produce();
        }

        // ---- S2-S3: [0]^(m) (Eq. 21) and Eq. 24 level by level for every primitive quartet; slot = kk*Kbra + kb ----
        {
            const int nR = g.Kbra * g.Kket;
            for (int it = tid; it < nR * (L + 1); it += NTHR) {
                const int s = it / (L + 1), m = it - s * (L + 1);
                const double *hbp = hdr + 4 * (s % g.Kbra), *hkp = hdr + 4 * (g.Kbra + s / g.Kbra);
                const double p = hbp[0], qq = hkp[0];
                const double X = hbp[1] - hkp[1], Y = hbp[2] - hkp[2], Z = hbp[3] - hkp[3];
                const double rho = p * qq / (p + qq);
                const double T = rho * (X * X + Y * Y + Z * Z);
                double f = 34.98683665524972497 / (p * qq * sqrt(p + qq)) * boys_single(m, T, g.boys_tab);   // 2 pi^{5/2}
                const double m2r = -2.0 * rho;
                for (int i = 0; i < m; ++i) f *= m2r;
                G0[s * (L + 1) + m] = f;
                if (m == L) ((L & 1) ? R1 + s * g.rs1 : R0 + s * g.rs0)[0] = f;
                if (m == 0) { PQ[3 * s] = X; PQ[3 * s + 1] = Y; PQ[3 * s + 2] = Z; }
            }
            __syncthreads();
            for (int m = L - 1; m >= 0; --m) {
                const int ne = nherm(L - m);
                for (int it = tid; it < nR * ne; it += NTHR) {
                    const int s = it / ne, e = it - s * ne;
                    const double *old = (m & 1) ? R0 + s * g.rs0 : R1 + s * g.rs1;
                    double *nw = (m & 1) ? R1 + s * g.rs1 : R0 + s * g.rs0;
                    const uint32_t w = __ldg(&lut[e].x);
                    double val;
                    if (e == 0) val = G0[s * (L + 1) + m];
                    else {
                        val = PQ[3 * s + (w >> 24 & 3)] * old[w & 0xfff];
                        const int cf = w >> 26;
                        if (cf) val = fma((double)cf, old[w >> 12 & 0xfff], val);
                    }
                    nw[e] = val;
                }
                __syncthreads();
            }
        }

        // ---- S4-S5 per cd tile ----
        for (int j = 0; j < g.ntile; ++j) {
            const int cd0 = j * NT;
            const int nnt = min(NW, (g.ncd - cd0 + 7) >> 3);
            double c2[MD_HL_MT2][NW][2];                       // the [ab|cd] tile, summed over the row blocks
#pragma unroll
            for (int t = 0; t < MD_HL_MT2; ++t)
#pragma unroll
                for (int n = 0; n < NW; ++n) c2[t][n][0] = c2[t][n][1] = 0.0;
            for (int blk = 0; blk < g.nblk; ++blk) {
            // GEMM1 (Eqs. 19, 25): rows = stacked (kb, p~) of the row block, columns = this cd tile, K = (kk, q~)
            // One row pass, specialised on the number of row tiles this warp really owns in it (the last pass is ragged):
            // no tensor-core step is spent on tiles past the end, and the inner loop stays branch-free.
            auto gemm1_pass = [&](auto mwc, int pass) {
                constexpr int MWc = decltype(mwc)::value, MWa = MWc > 0 ? MWc : 1;
                uint32_t wrow[MWa];
                int rbase[MWa];
#pragma unroll
                for (int i = 0; i < MWc; ++i) {
                    const int mt = (pass * MW + i) * NWARPS + warp;
                    const int2 ri = rowinfo[mt * 8 + lr];
                    wrow[i] = (uint32_t)ri.x; rbase[i] = min(blk * g.kbb + ri.y, g.Kbra - 1) * g.rs0;
                }
                double acc[MWa][NW][2];
#pragma unroll
                for (int i = 0; i < MWa; ++i)
#pragma unroll
                    for (int n = 0; n < NW; ++n) acc[i][n][0] = acc[i][n][1] = 0.0;
                for (int kk = 0; kk < g.Kket; ++kk) {
                    const double *Rk = R0 + (long long)kk * g.Kbra * g.rs0;
                    for (int c = c_first; c < nc1; ++c) {
                        const double *B = acquire() + lc * NTS + lr;
                        if (MWc > 0) {
                            const int q0 = c * MD_HL_KC1 + lc;
                            const int nsteps = min(MD_HL_KC1 / 4, (nhk - c * MD_HL_KC1 + 3) >> 2);   // rows >= nhk of Hk are zero
                            if (nsteps == MD_HL_KC1 / 4) {
                                uint32_t wq[MD_HL_KC1 / 4];
#pragma unroll
                                for (int k = 0; k < MD_HL_KC1 / 4; ++k) wq[k] = s_herm[min(q0 + 4 * k, nhk - 1)];
                                if (nnt == NW) {
#pragma unroll
                                    for (int k = 0; k < MD_HL_KC1 / 4; ++k)
                                        hl_gemm1_step<MWa, NW, true>(acc, B + 4 * k * NTS, Rk, rbase, wrow, wq[k], nnt);
                                } else {
#pragma unroll
                                    for (int k = 0; k < MD_HL_KC1 / 4; ++k)
                                        hl_gemm1_step<MWa, NW, false>(acc, B + 4 * k * NTS, Rk, rbase, wrow, wq[k], nnt);
                                }
                            } else {
                                for (int k = 0; k < nsteps; ++k)
                                    hl_gemm1_step<MWa, NW, false>(acc, B + 4 * k * NTS, Rk, rbase, wrow, s_herm[min(q0 + 4 * k, nhk - 1)], nnt);
                            }
                        }
                        release();
                    }
                }
#pragma unroll
                for (int i = 0; i < MWc; ++i) {
                    const int mt = (pass * MW + i) * NWARPS + warp;
#pragma unroll
                    for (int n = 0; n < NW; ++n)
                        *(double2 *)(Vp + (mt * 8 + lr) * NTS + n * 8 + 2 * lc) = make_double2(acc[i][n][0], acc[i][n][1]);
                }
            };
            for (int pass = 0; pass < npass; ++pass) {
                const int left_tiles = nmt - pass * MW * NWARPS - warp;      // this warp owns tiles warp, warp + NWARPS, .. of the pass
                const int mine = left_tiles <= 0 ? 0 : min(MW, (left_tiles + NWARPS - 1) / NWARPS);
                using std::integral_constant;
                if (mine == MW) gemm1_pass(integral_constant<int, MW>{}, pass);
                else if (MW > 3 && mine == 3) gemm1_pass(integral_constant<int, (MW > 3 ? 3 : 0)>{}, pass);
                else if (MW > 2 && mine == 2) gemm1_pass(integral_constant<int, (MW > 2 ? 2 : 0)>{}, pass);
                else if (MW > 1 && mine == 1) gemm1_pass(integral_constant<int, (MW > 1 ? 1 : 0)>{}, pass);
                else gemm1_pass(integral_constant<int, 0>{}, pass);
            }
            __syncthreads();
            // GEMM2 (Eq. 26): rows = ab (MD_HL_MT2 tiles per warp), columns = the cd tile, K = stacked (kb, p~)
            // specialised on the number of ab row tiles this warp owns (TC) and on a full cd tile: no guards inside
            auto gemm2 = [&](auto tc, auto full) {
                constexpr int TC = decltype(tc)::value;
                constexpr bool FULLN = decltype(full)::value;
                for (int c = 0; c < nc2; ++c) {
                    const double *A = acquire() + lc * g.sb + warp * 8 + lr;
                    const double *V = Vp + (c * g.kc2 + lc) * NTS + lr;
                    for (int u = 0; u < g.kc2; u += 8) {
#pragma unroll
                        for (int ks = 0; ks < 2; ++ks) {
                            double bfr[NW], a[TC > 0 ? TC : 1];
#pragma unroll
                            for (int n = 0; n < NW; ++n) bfr[n] = V[(u + ks * 4) * NTS + n * 8];
#pragma unroll
                            for (int t = 0; t < TC; ++t) a[t] = A[(u + ks * 4) * g.sb + t * NWARPS * 8];
#pragma unroll
                            for (int t = 0; t < TC; ++t)
#pragma unroll
                                for (int n = 0; n < NW; ++n)
                                    if (FULLN || n < nnt) hl_dmma884(c2[t][n][0], c2[t][n][1], a[t], bfr[n]);
                        }
                    }
                    release();
                }
            };
            {
                const int tc = max(0, (nmt2 - warp + NWARPS - 1) / NWARPS);
                using std::integral_constant;
                using T = std::true_type; using F = std::false_type;
                if (nnt == NW) {
                    if (tc >= 3) gemm2(integral_constant<int, 3>{}, T{});
                    else if (tc == 2) gemm2(integral_constant<int, 2>{}, T{});
                    else if (tc == 1) gemm2(integral_constant<int, 1>{}, T{});
                    else gemm2(integral_constant<int, 0>{}, T{});
                } else {
                    if (tc >= 3) gemm2(integral_constant<int, 3>{}, F{});
                    else if (tc == 2) gemm2(integral_constant<int, 2>{}, F{});
                    else if (tc == 1) gemm2(integral_constant<int, 1>{}, F{});
                    else gemm2(integral_constant<int, 0>{}, F{});
                }
            }
            if (blk + 1 < g.nblk) __syncthreads();             // [p~|cd] is rewritten by the next row block
            }
            // S5: the accumulators are the final [ab|cd] tile
#pragma unroll
            for (int t = 0; t < MD_HL_MT2; ++t) {
                const int ab = (warp + t * NWARPS) * 8 + lr;
                if (ab < g.nab) {
#pragma unroll
                    for (int n = 0; n < NW; ++n) {
                        const int cd = cd0 + n * 8 + 2 * lc;
                        double *o = out + ab * g.s_ab + cd * g.s_cd;
                        if (cd < g.ncd) o[0] = c2[t][n][0];
                        if (cd + 1 < g.ncd) o[g.s_cd] = c2[t][n][1];
                    }
                }
            }
            __syncthreads();                               // [p~|cd] is rewritten by the next tile
        }
    }
}

}  // namespace mdb
