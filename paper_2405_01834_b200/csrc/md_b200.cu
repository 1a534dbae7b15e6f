// md_b200.cu -- host side of the C ABI in include/md_b200.h: argument checks, workspace,
// variant selection and kernel launches.  No integral arithmetic runs on the host; the only
// host-computed numbers are the constant index / solid-harmonic coefficient tables uploaded
// once by md_init().
#include <algorithm>
#include <cmath>
#include <cstdio>
#include <cstdlib>
#include <cstring>
#include <mutex>
#include <vector>

#include "../../include/md_b200.h"
#include "boys.cuh"
#include "common.cuh"
#include "fused_api.cuh"
#include "generic.cuh"
#include "hl_api.cuh"
#include "lowl_api.cuh"
#include "eri3s_api.cuh"
#include "mma_api.cuh"
#include "pair.cuh"
#include "warp.cuh"
#include "peak.cuh"

using namespace mdb;

#define MD_LOWL_KMAX (1 << 24)   // by measurement the one-thread-per-quartet kernel wins at every contraction degree tried (K = 1..6 per shell)

namespace {

struct State {
    bool init = false;
    int device = -1;
    double *boys_tab = nullptr;
    void *user_ws = nullptr;     // caller-owned workspace (md_set_workspace)
    size_t user_bytes = 0;
    int variant = MD_VARIANT_AUTO;
    int last_variant = 0;
    int last_launches = 0;
    int last_mma_info[8] = {0};
    int last_f2_info[8] = {0};
    int last_hl_info[8] = {0};
    int nsm = 148;
    int max_smem = 227 * 1024;
    char cuda_err[256] = "";
    void *static_ws = nullptr;   // device address of g_static_scratch (md_eri4_static), resolved in md_init
} S;

// Scratch of md_eri4_static (include/md_b200.h): pair records of the runtime-l chain for callers that must not allocate.
// In host code this name is only a handle for cudaGetSymbolAddress (md_init), never a device address.
static __device__ __align__(256) unsigned char g_static_scratch[MD_STATIC_SCRATCH_BYTES];

// Measured-best variant per (canonical class, contracted or not), written by `python bench.py --sweep autotune` on one
// B200 for the independent-quartet structure (profiles/r02_autotune.md) and checked in.  Classes that are missing, and calls the
// table cannot describe (paper layout, huge per-pair records, the product-mode exceptions), follow the rules in run().
struct VariantRow { signed char la, lb, lc, ld, three, contracted, variant; };
const VariantRow g_variant_table[] = {
#include "variant_table.inc"
    {-1, -1, -1, -1, 0, 0, 0}};

int table_variant(int la, int lb, int lc, int ld, bool three, bool contracted) {
    if (la < lb) std::swap(la, lb);
    if (!three && lc < ld) std::swap(lc, ld);
    if (!three && (la < lc || (la == lc && lb < ld))) { std::swap(la, lc); std::swap(lb, ld); }   // bra >= ket (sweep 6 order)
    for (const VariantRow *r = g_variant_table; r->la >= 0; ++r)
        if (r->la == la && r->lb == lb && r->lc == lc && r->ld == ld && (r->three != 0) == three && (r->contracted != 0) == contracted)
            return r->variant;
    return 0;
}

int cuda_fail(cudaError_t e) {
    snprintf(S.cuda_err, sizeof(S.cuda_err), "%s", cudaGetErrorString(e));
    return MD_ECUDA;
}
#define CK(call) do { cudaError_t e_ = (call); if (e_ != cudaSuccess) return cuda_fail(e_); } while (0)

// Cartesian -> Racah-normalised real solid harmonic coefficients (Eqs. 16-17;
// formula: DESIGN.md reading O2, the textbook expansion of the paper's Ref. 29):
//   S_lm = N_lm sum_t sum_u sum_w C x^{2t+|m|-2u-w} y^{2u+w} z^{l-2t-|m|},  w even (m>=0) / odd (m<0)
//   C = (-1)^{t+(w-w0)/2} 4^{-t} binom(l,t) binom(l-t,|m|+t) binom(t,u) binom(|m|,w)
//   N_lm = sqrt(2 (l+|m|)! (l-|m|)! / 2^{delta_m0}) / (2^{|m|} l!)
void make_tables(std::vector<uint32_t> &herm, std::vector<double> &solid) {
    herm.clear();
    for (int n = 0; n <= MD_LTOT; ++n)
        for (int t = n; t >= 0; --t)
            for (int u = n - t; u >= 0; --u) herm.push_back(t | (u << 8) | ((n - t - u) << 16) | (n << 24));
    auto fact = [](int n) { long double r = 1; for (int i = 2; i <= n; ++i) r *= i; return r; };
    auto binom = [&](int n, int k) -> long double { return (k < 0 || k > n) ? 0.0L : fact(n) / (fact(k) * fact(n - k)); };
    solid.assign(MD_SOLID_TOTAL, 0.0);
    for (int l = 0; l <= MD_LMAX; ++l) {
        double *C = solid.data() + solid_off(l);
        const int nc = ncart(l);
        for (int m = -l; m <= l; ++m) {
            const int am = std::abs(m), w0 = m < 0 ? 1 : 0;
            long double N = sqrtl(2.0L * fact(l + am) * fact(l - am) / (m == 0 ? 2.0L : 1.0L)) / (powl(2.0L, am) * fact(l));
            for (int t = 0; 2 * t + am <= l; ++t)
                for (int u = 0; u <= t; ++u)
                    for (int w = w0; w <= am; w += 2) {
                        long double c = powl(0.25L, t) * binom(l, t) * binom(l - t, am + t) * binom(t, u) * binom(am, w);
                        if ((t + (w - w0) / 2) & 1) c = -c;
                        int ex = 2 * t + am - 2 * u - w, ey = 2 * u + w;
                        int k = herm_index(ex, ey, l - ex - ey) - nherm(l - 1);
                        C[(m + l) * nc + k] += (double)(N * c);
                    }
        }
    }
}

int check_shells(const md_shells *s) {
    if (!s) return MD_EINVAL;
    if (s->l < 0 || s->l > MD_MAX_L || s->K < 1 || s->K > MD_MAX_K || s->n < 0) return MD_EINVAL;
    if (s->n > 0 && (!s->center || !s->exps || !s->coefs)) return MD_EINVAL;
    return MD_OK;
}
int check_pairs(const md_pairs *p) {
    if (!p || p->npairs < 0) return MD_EINVAL;
    int e = check_shells(&p->a);
    if (e) return e;
    e = check_shells(&p->b);
    if (e) return e;
    if (!p->idx && (p->npairs > p->a.n || p->npairs > p->b.n)) return MD_EINVAL;
    return MD_OK;
}

ShellView view(const md_shells &s) { return ShellView{s.center, s.exps, s.coefs, s.l, s.K}; }
PairView view(const md_pairs &p) { return PairView{view(p.a), view(p.b), p.idx, p.npairs, 0}; }
PairView view_single(const md_shells &x) { return PairView{view(x), view(x), nullptr, x.n, 1}; }

struct Shape {
    int la, lb, lc, ld, Ka, Kb, Kc, Kd;
    int nab, ncd, nhb, nhk;
    long long stride_b, stride_k;
};
Shape shape_of(const PairView &b, const PairView &k, int pure) {
    Shape s;
    s.la = b.a.l; s.lb = b.single ? 0 : b.b.l; s.lc = k.a.l; s.ld = k.single ? 0 : k.b.l;
    s.Ka = b.a.K; s.Kb = b.single ? 1 : b.b.K; s.Kc = k.a.K; s.Kd = k.single ? 1 : k.b.K;
    s.nab = ncomp(s.la, pure) * ncomp(s.lb, pure);
    s.ncd = ncomp(s.lc, pure) * ncomp(s.ld, pure);
    s.nhb = nherm(s.la + s.lb); s.nhk = nherm(s.lc + s.ld);
    s.stride_b = 4 + (long long)s.nhb * s.nab; s.stride_b += s.stride_b & 1;
    s.stride_k = 4 + (long long)s.nhk * s.ncd; s.stride_k += s.stride_k & 1;
    return s;
}
size_t generic_ws_bytes(const PairView &b, const PairView &k, int pure) {
    Shape s = shape_of(b, k, pure);
    return 8 * ((size_t)b.npairs * s.Ka * s.Kb * s.stride_b + (size_t)k.npairs * s.Kc * s.Kd * s.stride_k);
}

// Per-call scratch (pair data is computed per call and never kept).  Without a caller buffer the block is
// taken from the CUDA stream-ordered pool on the call's own stream and released there after the last launch, so calls
// in flight on different streams never share scratch and nothing synchronises.  In `dry` mode nothing is allocated or
// launched: the first request records its size and the call unwinds with MD_DRY (the *_workspace_bytes queries).
#define MD_DRY 2
struct Scratch {
    cudaStream_t st = nullptr;
    void *owned = nullptr;
    bool dry = false;
    size_t need = 0;
    int get(size_t bytes, void **out) {
        need = bytes;
        if (dry) return MD_DRY;
        if (bytes == 0) { *out = nullptr; return MD_OK; }
        if (S.user_ws) {
            if (bytes > S.user_bytes) return MD_ENOMEM;
            *out = S.user_ws;
            return MD_OK;
        }
        CK(cudaMallocAsync(&owned, bytes, st));
        *out = owned;
        return MD_OK;
    }
    void release() {
        if (owned) cudaFreeAsync(owned, st);
        owned = nullptr;
    }
};
// Every class with all l <= 2 has a first-generation fused kernel (fused_inst.cu), which needs no scratch.
bool fused_has_class(const PairView &b, const PairView &k) {
    return b.a.l <= 2 && (b.single || b.b.l <= 2) && k.a.l <= 2 && (k.single || k.b.l <= 2);
}
int scratch_get(void *ctx, size_t bytes, void **out) { return ((Scratch *)ctx)->get(bytes, out); }

__global__ void iota2_kernel(int32_t *idx, long long n) {
    const long long i = blockIdx.x * (long long)blockDim.x + threadIdx.x;
    if (i < n) { idx[2 * i] = (int32_t)i; idx[2 * i + 1] = (int32_t)i; }
}

int launch_pair_setup(const PairView &pv, int pure, int ket_sign, long long stride, double *rec, cudaStream_t st,
                      const int32_t *by_quartet = nullptr, long long q0 = 0, long long nrec = -1) {
    const int la = pv.a.l, lb = pv.single ? 0 : pv.b.l;
    const int Kab = pv.a.K * (pv.single ? 1 : pv.b.K);
    if (pv.npairs == 0 || nrec == 0) return MD_OK;
    PairSetupArgs a;
    a.pv = pv; a.pure = pure; a.ket_sign = ket_sign; a.stride = stride; a.rec = rec;
    a.by_quartet = by_quartet; a.q0 = q0; a.side = ket_sign;
    if (nrec >= 0) a.pv.npairs = nrec;
    const int esz = (la + 1) * (lb + 1) * (la + lb + 1);
    const int rowsz = ncart(la) * nsolid(lb);
    a.pchunk = std::max(1, std::min(nherm(la + lb), 4096 / rowsz));
    size_t smem = 8 * ((size_t)3 * esz + (pure ? (size_t)a.pchunk * rowsz : 0));
    long long nblk = a.pv.npairs * Kab;
    if (nblk > 0x7fffffffLL) return MD_EINVAL;
    switch (std::max(la, lb)) {
        case 0: pair_setup_kernel<0><<<(unsigned)nblk, 128, smem, st>>>(a); break;
        case 1: pair_setup_kernel<1><<<(unsigned)nblk, 128, smem, st>>>(a); break;
        case 2: pair_setup_kernel<2><<<(unsigned)nblk, 128, smem, st>>>(a); break;
        case 3: pair_setup_kernel<3><<<(unsigned)nblk, 128, smem, st>>>(a); break;
        case 4: pair_setup_kernel<4><<<(unsigned)nblk, 128, smem, st>>>(a); break;
        case 5: pair_setup_kernel<5><<<(unsigned)nblk, 128, smem, st>>>(a); break;
        default: pair_setup_kernel<6><<<(unsigned)nblk, 128, smem, st>>>(a); break;
    }
    S.last_launches++;
    CK(cudaGetLastError());
    return MD_OK;
}

// Output strides for both layouts (include/md_b200.h).
void out_strides(int layout, bool list_mode, long long nbra, long long nket, int nab, int ncd,
                 long long &s_q, long long &s_bi, long long &s_ki, long long &s_ab, long long &s_cd) {
    if (layout == MD_LAYOUT_PAPER) {           // out[ij + nbra*(ab + N_ab*(cd + N_cd*kl))]
        s_q = 0; s_bi = 1; s_ab = nbra; s_cd = nbra * nab; s_ki = nbra * (long long)nab * ncd;
    } else {
        s_ab = ncd; s_cd = 1;
        if (list_mode) { s_q = (long long)nab * ncd; s_bi = 0; s_ki = 0; }
        else { s_q = 0; s_bi = nket * (long long)nab * ncd; s_ki = (long long)nab * ncd; }
    }
}

int run_generic_once(const PairView &b, const PairView &k, long long nq, const int32_t *qidx, int pure, int layout,
                     double *out, cudaStream_t st, bool use_mma, Scratch &sc, void *ws, const int32_t *by_quartet, long long q0);

// Per-pair records grow with the pair batch (527 KB per (ff| pair at K = 4); a quartet LIST whose records would exceed
// MD_GEN_WS_BYTES is cut into chunks of quartets: records per quartet side (pair setup indexed by quartet), an identity
// index list for the quartet kernel, the same scratch reused by every chunk.
#define MD_GEN_WS_BYTES ((size_t)4 << 30)
int run_generic(const PairView &b, const PairView &k, long long nq, const int32_t *qidx, int pure, int layout,
                double *out, cudaStream_t st, bool use_mma, Scratch &sc) {
    const size_t full = generic_ws_bytes(b, k, pure);
    if (full <= MD_GEN_WS_BYTES || !qidx || layout != MD_LAYOUT_QUARTET_MAJOR) {
        void *ws = nullptr;
        int e = sc.get(full, &ws);
        if (e) return e;
        return run_generic_once(b, k, nq, qidx, pure, layout, out, st, use_mma, sc, ws, nullptr, 0);
    }
    Shape s = shape_of(b, k, pure);
    const size_t per = 8 * ((size_t)s.Ka * s.Kb * s.stride_b + (size_t)s.Kc * s.Kd * s.stride_k) + 2 * sizeof(int32_t);
    const long long chunk = std::max<long long>(1, std::min<long long>(nq, (long long)(MD_GEN_WS_BYTES / per)));
    void *ws = nullptr;
    int e = sc.get((size_t)chunk * per, &ws);
    if (e) return e;
    int32_t *iota = (int32_t *)((char *)ws + (size_t)chunk * (per - 2 * sizeof(int32_t)));
    iota2_kernel<<<(unsigned)((chunk + 255) / 256), 256, 0, st>>>(iota, chunk);
    int launches = 1;
    PairView bc = b, kc = k;
    bc.npairs = chunk; kc.npairs = chunk;
    for (long long q0 = 0; q0 < nq; q0 += chunk) {
        const long long m = std::min(chunk, nq - q0);
        bc.npairs = m; kc.npairs = m;
        S.last_launches = 0;
        e = run_generic_once(bc, kc, m, iota, pure, layout, out + q0 * (long long)s.nab * s.ncd, st, use_mma, sc, ws, qidx, q0);
        launches += S.last_launches;
        if (e) return e;
    }
    S.last_launches = launches;
    return MD_OK;
}

int run_generic_once(const PairView &b, const PairView &k, long long nq, const int32_t *qidx, int pure, int layout,
                     double *out, cudaStream_t st, bool use_mma, Scratch &sc, void *ws, const int32_t *by_quartet, long long q0) {
    Shape s = shape_of(b, k, pure);
    int e;
    (void)sc;
    double *rec_b = (double *)ws;
    double *rec_k = rec_b + (size_t)b.npairs * s.Ka * s.Kb * s.stride_b;
    if ((e = launch_pair_setup(b, pure, 0, s.stride_b, rec_b, st, by_quartet, q0, by_quartet ? nq : -1))) return e;
    if ((e = launch_pair_setup(k, pure, 1, s.stride_k, rec_k, st, by_quartet, q0, by_quartet ? nq : -1))) return e;

    GenericArgs g;
    g.rec_bra = rec_b; g.rec_ket = rec_k; g.stride_bra = s.stride_b; g.stride_ket = s.stride_k;
    g.Kbra = s.Ka * s.Kb; g.Kket = s.Kc * s.Kd;
    g.Lb = s.la + s.lb; g.Lk = s.lc + s.ld; g.nab = s.nab; g.ncd = s.ncd;
    g.qidx = qidx; g.nq = nq; g.nket = k.npairs; g.out = out; g.boys_tab = S.boys_tab;
    out_strides(layout, qidx != nullptr, b.npairs, k.npairs, s.nab, s.ncd, g.s_q, g.s_bi, g.s_ki, g.s_ab, g.s_cd);
    const int Sd = g.Lb + g.Lk + 1;
    size_t fixed = 8 * ((size_t)Sd * Sd * Sd + Sd + 2) + 4 * (size_t)(s.nhb + s.nhk) + 64;
    size_t budget = (size_t)S.max_smem - 1024;
    long long ct = ((long long)budget - (long long)fixed) / (8LL * s.nhb);
    if (ct < 1) return MD_EINVAL;
    // a modest tile keeps several CTAs resident for the small classes
    ct = std::min<long long>(ct, std::max(16, 4096 / s.nhb));
    g.ct = (int)std::min<long long>(ct, s.ncd);
    size_t smem = fixed + 8 * (size_t)s.nhb * g.ct;
    // Small classes: one warp per quartet (warp.cuh) instead of one CTA per quartet.
    const int kq0 = (k.single && pure) ? nherm(k.a.l - 1) : 0;
    if (use_mma && S.variant != MD_VARIANT_MMA && g.Lb + g.Lk <= MD_WARP_LMAX && s.nhb * s.ncd <= MD_WARP_HALF) {
        WarpArgs w;
        w.rec_bra = rec_b; w.rec_ket = rec_k; w.stride_bra = s.stride_b; w.stride_ket = s.stride_k;
        w.Kbra = g.Kbra; w.Kket = g.Kket; w.Lb = g.Lb; w.Lk = g.Lk; w.nab = s.nab; w.ncd = s.ncd; w.kq0 = kq0;
        w.qidx = qidx; w.nq = nq; w.nket = k.npairs; w.out = out;
        w.s_q = g.s_q; w.s_bi = g.s_bi; w.s_ki = g.s_ki; w.s_ab = g.s_ab; w.s_cd = g.s_cd;
        w.boys_tab = S.boys_tab; w.rlut = fused_rlut();
        const size_t wsm = 8 * (size_t)(MD_WARP_THREADS / 32) * warp_smem_doubles(g.Lb + g.Lk, s.nhb, s.ncd);
        const long long nblk = (nq + MD_WARP_THREADS / 32 - 1) / (MD_WARP_THREADS / 32);
        const unsigned wgrid = (unsigned)std::min<long long>(nblk, (long long)S.nsm * 8);
        eri_warp_kernel<<<wgrid, MD_WARP_THREADS, wsm, st>>>(w);
        S.last_launches++;
        CK(cudaGetLastError());
        S.last_variant = MD_VARIANT_WARP;
        return MD_OK;
    }
    if (use_mma) {
        MmaCall c;
        c.rec_bra = rec_b; c.rec_ket = rec_k; c.stride_bra = s.stride_b; c.stride_ket = s.stride_k;
        c.Kbra = g.Kbra; c.Kket = g.Kket; c.Lb = g.Lb; c.Lk = g.Lk; c.nab = s.nab; c.ncd = s.ncd;
        // one-centre solid ket (Hobson, pair.cuh): Hermite rows of order < l_X are exactly zero
        c.kq0 = (k.single && pure) ? nherm(k.a.l - 1) : 0;
        c.qidx = qidx; c.nq = nq; c.nket = k.npairs; c.out = out;
        c.s_q = g.s_q; c.s_bi = g.s_bi; c.s_ki = g.s_ki; c.s_ab = g.s_ab; c.s_cd = g.s_cd;
        c.boys_tab = S.boys_tab; c.rlut = fused_rlut();
        const cudaError_t me = mma_launch(c, S.nsm, st, S.last_mma_info);
        if (me == cudaSuccess) {
            S.last_launches++;
            S.last_variant = MD_VARIANT_MMA;
            return MD_OK;
        }
        if (me != cudaErrorInvalidConfiguration) return cuda_fail(me);
        // no DMMA tile shape fits shared memory for this (class, K): the DFMA kernel below serves every class
    }
    unsigned grid = (unsigned)std::min<long long>(nq, (long long)S.nsm * 8);
    eri_generic_kernel<<<grid, MD_GEN_THREADS, smem, st>>>(g);
    S.last_launches++;
    CK(cudaGetLastError());
    S.last_variant = MD_VARIANT_GENERIC;
    return MD_OK;
}

int run_rules(const PairView &b, const PairView &k, long long nq, const int32_t *qidx, int pure, int layout,
              double *out, long long cap, cudaStream_t st, Scratch &sc) {
    if (pure != 0 && pure != 1) return MD_EINVAL;
    if (layout != MD_LAYOUT_QUARTET_MAJOR && layout != MD_LAYOUT_PAPER) return MD_EINVAL;
    if (layout == MD_LAYOUT_PAPER && qidx) return MD_EINVAL;
    if (nq < 0) return MD_EINVAL;
    if (!qidx && nq != b.npairs * k.npairs) return MD_EINVAL;
    Shape s = shape_of(b, k, pure);
    if (!sc.dry && (long long)s.nab * s.ncd * nq > cap) return MD_ECAPACITY;
    if (!sc.dry && nq > 0 && !out) return MD_EINVAL;
    int e = md_init();
    if (e) return e;
    S.last_launches = 0;
    if (nq == 0) return MD_OK;
    // Measured exception: a bra x ket PRODUCT with an s-type ket ((dd|ss), (dd|s)) amortises pair
    // setup over the whole ket list, and the one-warp-per-quartet kernel is then 2-3.5x faster than the fused one.
    const bool product_s_ket = S.variant == MD_VARIANT_AUTO && !qidx && k.a.l == 0 && (k.single || k.b.l == 0) &&
                               b.a.l + (b.single ? 0 : b.b.l) >= 4 && nq >= 8 * (b.npairs + k.npairs);
    if (product_s_ket) return run_generic(b, k, nq, qidx, pure, layout, out, st, true, sc);
    // Every l <= 1, quartet-major output: one thread per quartet, registers only, coalesced tile stores (lowl.cuh).  By
    // measurement (profiles/r02_autotune.csv) it wins while the primitive loop is short; long contractions stay with the fused kernels.
    if ((S.variant == MD_VARIANT_LOWL || (S.variant == MD_VARIANT_AUTO && (long long)s.Ka * s.Kb * s.Kc * s.Kd <= MD_LOWL_KMAX)) &&
        layout == MD_LAYOUT_QUARTET_MAJOR && lowl_has_class(b, k)) {
        if (sc.dry) { sc.need = 0; return MD_DRY; }
        if (lowl_dispatch(b, k, nq, qidx, pure, out, S.boys_tab, S.nsm, st) == 1) {
            S.last_launches++;
            CK(cudaGetLastError());
            S.last_variant = MD_VARIANT_LOWL;
            return MD_OK;
        }
    }
    // 3-center with la, lb <= 3 (BASELINE configs[2]): one warp per triplet in the sparse Cartesian form (eri3s.cuh); by
    // measurement (profiles/r02_autotune.csv) under AUTO when a shell has l >= 3 or la + lb >= 4; the smaller l <= 2 classes stay with `fused`
    // ((ds|d) 0.097 against 0.379 ms per 100,000).
    // The same kernel serves 4-center classes with an s shell second in one pair, (ab|c s) or (a s|cd); those only when the
    // table (or the caller) names it.
    if ((S.variant == MD_VARIANT_ERI3S || (S.variant == MD_VARIANT_AUTO && k.single && (std::max({s.la, s.lb, s.lc}) >= 3 || s.la + s.lb >= 4))) &&
        layout == MD_LAYOUT_QUARTET_MAJOR && eri3s_has_class(b, k)) {
        if (sc.dry) { sc.need = 0; return MD_DRY; }
        if (eri3s_dispatch(b, k, nq, qidx, pure, out, S.boys_tab, fused_rlut(), S.nsm, st) == 1) {
            S.last_launches++;
            CK(cudaGetLastError());
            S.last_variant = MD_VARIANT_ERI3S;
            return MD_OK;
        }
    }
    if (S.variant == MD_VARIANT_AUTO || S.variant == MD_VARIANT_FUSED2) {
        // By measurement (profiles/r01_sweep_l2.md, r02_autotune.csv): the warp-specialised kernel wins on every instantiated class
        // once the primitive loop is long enough to fill its pipeline, and on (dd|dd) for any K.
        const long long nprim = (long long)b.a.K * (b.single ? 1 : b.b.K) * k.a.K * (k.single ? 1 : k.b.K);
        const bool dddd = b.a.l == 2 && !b.single && b.b.l == 2 && k.a.l == 2 && !k.single && k.b.l == 2;
        if (S.variant == MD_VARIANT_FUSED2 || nprim >= 4 || (dddd && nq >= 150000)) {
            int r = fused2_dispatch(b, k, nq, qidx, pure, layout, out, S.boys_tab, S.nsm, st, S.last_f2_info, scratch_get, &sc);
            if (r == 1) {
                S.last_launches++;
                CK(cudaGetLastError());
                S.last_variant = MD_VARIANT_FUSED2;
                return MD_OK;
            }
            if (r == MD_DRY) return r;
            // under AUTO a caller buffer too small for the pair tables falls through to the first fused kernel (no scratch)
            if (r < 0 && !(r == MD_ENOMEM && S.variant == MD_VARIANT_AUTO)) return r;
        }
    }
    if (S.variant == MD_VARIANT_AUTO || S.variant == MD_VARIANT_FUSED || S.variant == MD_VARIANT_FUSED2) {
        if (sc.dry && fused_has_class(b, k)) { sc.need = 0; return MD_DRY; }
        int r = fused_dispatch(b, k, nq, qidx, pure, layout, out, S.boys_tab, S.nsm, st, S.variant == MD_VARIANT_FUSED);
        if (r == 1) {
            S.last_launches++;
            CK(cudaGetLastError());
            S.last_variant = MD_VARIANT_FUSED;
            return MD_OK;
        }
        if (r < 0) return r;
    }
    if (S.variant == MD_VARIANT_AUTO || S.variant == MD_VARIANT_HL) {
        // Classes with an l >= 3 shell: the one-launch high-l kernel (hl.cuh) when its tiles fit the (class, K).
        HlCall c;
        c.bra = b; c.ket = k; c.pure = pure; c.qidx = qidx; c.nq = nq; c.out = out;
        out_strides(layout, qidx != nullptr, b.npairs, k.npairs, s.nab, s.ncd, c.s_q, c.s_bi, c.s_ki, c.s_ab, c.s_cd);
        c.boys_tab = S.boys_tab; c.rlut = fused_rlut();
        size_t need = 0;
        // By measurement (profiles/r02_autotune.csv): the one-launch kernel wins from (gg|gg) upward (N~_bra N~_ket >= 16,000:
        // (gg|gg) 27,225, (fg|hi) 43,680); below that ((ff|ff) 7,056, (ff|i) 7,056) its per-quartet phases are too short
        // to fill a CTA and pair setup + the runtime-l kernels are faster.
        const bool large = (long long)s.nhb * s.nhk >= 16000;
        if ((S.variant == MD_VARIANT_HL || large) && hl_plan(c, S.nsm, &need)) {
            void *ws = nullptr;
            int e = sc.get(need, &ws);
            if (e) return e;
            int nl = 0;
            CK(hl_launch(c, S.nsm, ws, st, S.last_hl_info, &nl));
            S.last_launches += nl;
            S.last_variant = MD_VARIANT_HL;
            return MD_OK;
        }
    }
    return run_generic(b, k, nq, qidx, pure, layout, out, st, S.variant != MD_VARIANT_GENERIC, sc);
}

// AUTO: the checked-in table first (a forced variant for this one call), then the rules.
int run(const PairView &b, const PairView &k, long long nq, const int32_t *qidx, int pure, int layout,
        double *out, long long cap, cudaStream_t st, Scratch &sc) {
    if (S.variant != MD_VARIANT_AUTO || (pure != 0 && pure != 1) || getenv("MD_NO_TABLE")) return run_rules(b, k, nq, qidx, pure, layout, out, cap, st, sc);
    const Shape s = shape_of(b, k, pure);
    const bool product_mode = !qidx && nq > 1;
    int tv = 0;
    if (!product_mode && layout == MD_LAYOUT_QUARTET_MAJOR && !b.single)
        tv = table_variant(s.la, s.lb, s.lc, s.ld, k.single != 0, (long long)s.Ka * s.Kb * s.Kc * s.Kd > 1);
    // The table was measured on independent quartets, where every quartet pays its own pair setup.  The one-warp kernel's
    // 4-center form recomputes its 1-D tables per quartet; when pairs are shared by many quartets (a screened molecule list) the
    // kernels that read per-pair records win that case back (1.3e8 against about 5e7 quartets/s on (fd|ds)), so the rules decide.
    if (tv == MD_VARIANT_ERI3S && !k.single && nq >= 8 * (b.npairs + k.npairs)) tv = 0;
    if (!tv) return run_rules(b, k, nq, qidx, pure, layout, out, cap, st, sc);
    S.variant = tv;
    int e = run_rules(b, k, nq, qidx, pure, layout, out, cap, st, sc);
    S.variant = MD_VARIANT_AUTO;
    if (e == MD_ENOMEM) e = run_rules(b, k, nq, qidx, pure, layout, out, cap, st, sc);   // caller buffer too small for the table's choice
    return e;
}

int run_call(const PairView &b, const PairView &k, long long nq, const int32_t *qidx, int pure, int layout,
             double *out, long long cap, cudaStream_t st) {
    Scratch sc;
    sc.st = st;
    const int e = run(b, k, nq, qidx, pure, layout, out, cap, st, sc);
    sc.release();                                   // stream-ordered: after the kernels enqueued above
    return e;
}
long long run_query(const PairView &b, const PairView &k, long long nq, int list_mode, int pure) {
    Scratch sc;
    sc.dry = true;
    static const int32_t dummy[2] = {0, 0};        // only its non-NULL-ness is looked at in dry mode
    const int e = run(b, k, nq, list_mode ? dummy : nullptr, pure, MD_LAYOUT_QUARTET_MAJOR, nullptr, 0, nullptr, sc);
    if (e == MD_DRY) return (long long)sc.need;
    return e < 0 ? e : 0;                           // MD_OK: nothing to do (nq == 0)
}


// ---- exchange digestion for classes without an in-kernel epilogue: [ab|cd] of a chunk of quartets goes to an L2-sized
// scratch (never the full V of PAPER.md Eq. 33) and is contracted by this kernel (Eqs. 34-35: atomic reduction into K).
__global__ void product_idx_kernel(int32_t *idx, long long q0, long long n, long long nket) {
    const long long i = blockIdx.x * (long long)blockDim.x + threadIdx.x;
    if (i < n) { idx[2 * i] = (int32_t)((q0 + i) / nket); idx[2 * i + 1] = (int32_t)((q0 + i) % nket); }
}
__global__ void __launch_bounds__(128) exchange_digest_kernel(const double *V, long long nq, const int32_t *qidx,
                                                              const int32_t *bidx, const int32_t *kidx, int na, int nb, int nc,
                                                              int nd, const int32_t *off_a, const int32_t *off_b,
                                                              const int32_t *off_c, const int32_t *off_d, long long n,
                                                              const double *D, double *K) {
    for (long long q = blockIdx.x; q < nq; q += gridDim.x) {
        const long long bi = qidx[2 * q], ki = qidx[2 * q + 1];
        const long long ia = bidx ? bidx[2 * bi] : bi, ib = bidx ? bidx[2 * bi + 1] : bi;
        const long long ic = kidx ? kidx[2 * ki] : ki, id = kidx ? kidx[2 * ki + 1] : ki;
        const long long oa = off_a[ia], ob = off_b[ib], oc = off_c[ic], od = off_d[id];
        const double *v = V + q * (long long)na * nb * nc * nd;
        for (int t = threadIdx.x; t < nb * nc; t += blockDim.x) {
            const int b = t / nc, c = t - b * nc;
            double s = 0.0;
            for (int a = 0; a < na; ++a) {
                const double *row = v + (((long long)a * nb + b) * nc + c) * nd;
                const double *dr = D + (oa + a) * n + od;
                for (int d = 0; d < nd; ++d) s = fma(row[d], dr[d], s);
            }
            atomicAdd(K + (ob + b) * n + oc + c, s);
        }
    }
}

int run_exchange(const md_pairs *bra, const md_pairs *ket, long long nq, const int32_t *qidx, int pure, const int32_t *const off[4],
                 long long nao, const double *D, double *K, cudaStream_t st) {
    const PairView b = view(*bra), k = view(*ket);
    if (nq == 0) return MD_OK;
    if (!qidx && nq != b.npairs * k.npairs) return MD_EINVAL;
    S.last_launches = 0;
    if (fused_has_class(b, k)) {                                  // every l <= 2: digestion in the kernel epilogue, no V at all
        FusedDigest dg{K, D, nao, {off[0], off[1], off[2], off[3]}};
        int r = fused_dispatch(b, k, nq, qidx, pure, MD_LAYOUT_QUARTET_MAJOR, nullptr, S.boys_tab, S.nsm, st, true, &dg);
        if (r == 1) {
            S.last_launches++;
            CK(cudaGetLastError());
            S.last_variant = MD_VARIANT_FUSED;
            return MD_OK;
        }
        if (r < 0) return r;
    }
    const int na = ncomp(b.a.l, pure), nb = ncomp(b.b.l, pure), nc = ncomp(k.a.l, pure), nd = ncomp(k.b.l, pure);
    const long long per = (long long)na * nb * nc * nd;
    const long long chunk = std::max<long long>(1, std::min<long long>(nq, ((long long)48 << 20) / (8 * per)));   // V chunk stays in L2
    double *V = nullptr;
    int32_t *ci = nullptr;
    CK(cudaMallocAsync(&V, (size_t)chunk * per * 8, st));
    CK(cudaMallocAsync(&ci, (size_t)chunk * 2 * sizeof(int32_t), st));
    int e = MD_OK, launches = 0;
    for (long long q0 = 0; q0 < nq && e == MD_OK; q0 += chunk) {
        const long long m = std::min(chunk, nq - q0);
        const int32_t *qi = qidx ? qidx + 2 * q0 : ci;
        if (!qidx) { product_idx_kernel<<<(unsigned)((m + 255) / 256), 256, 0, st>>>(ci, q0, m, k.npairs); ++launches; }
        e = run_call(b, k, m, qi, pure, MD_LAYOUT_QUARTET_MAJOR, V, m * per, st);
        launches += S.last_launches;
        if (e == MD_OK) {
            exchange_digest_kernel<<<(unsigned)std::min<long long>(m, (long long)S.nsm * 16), 128, 0, st>>>(
                V, m, qi, b.idx, k.idx, na, nb, nc, nd, off[0], off[1], off[2], off[3], nao, D, K);
            ++launches;
        }
    }
    cudaFreeAsync(ci, st);
    cudaFreeAsync(V, st);
    S.last_launches = launches;
    if (e == MD_OK) CK(cudaGetLastError());
    return e;
}

// ---- first geometric derivatives ----------------------------------------------------
// A primitive Cartesian Gaussian (Eq. 1) depends on its centre A only through r - A:
//     d/dA_i G_a = 2 zeta G_{a+1_i} - a_i G_{a-1_i}.
// The derivative of (ab|cd) with respect to the centre of one shell is therefore the Cartesian integral batch with that
// shell RAISED (l + 1, coefficients 2 zeta_k c_k) minus a_i times the batch with the shell LOWERED (l - 1).  Both batches come
// from the integral kernels above (whatever variant the class selects); the kernels below form the coefficients, combine
// the two batches component by component, and apply the solid-harmonic transform (Eq. 16, linear and centre-independent)
// to the four indices afterwards.  A chunk of quartets at a time, so that the intermediates stay L2-sized.
__global__ void grad_coefs_kernel(const double *exps, const double *coefs, double *out, long long n) {
    const long long i = blockIdx.x * (long long)blockDim.x + threadIdx.x;
    if (i < n) out[i] = 2.0 * exps[i] * coefs[i];
}
// position of the Cartesian component with exponents (., ay, az) inside its shell (include/md_b200.h: ax descending, then ay)
__device__ __forceinline__ int grad_cart_pos(int ay, int az) { const int i = ay + az; return ((i * (i + 1)) >> 1) + az; }

// G[q][i][pre][k][post] = U[q][pre][k + 1_i][post] - k_i Dn[q][pre][k - 1_i][post]; k runs over the Cartesian components of
// the differentiated shell (angular momentum l), pre / post over the components of the shells before / after it.
__global__ void grad_combine_kernel(const double *__restrict__ U, const double *__restrict__ Dn, double *__restrict__ G,
                                    long long nq, int l, int pre, int post) {
    const int nk = ncart(l), nu = ncart(l + 1), nd = l > 0 ? ncart(l - 1) : 0;
    const long long per = (long long)pre * nk * post, total = nq * 3 * per;
    for (long long t = blockIdx.x * (long long)blockDim.x + threadIdx.x; t < total; t += (long long)gridDim.x * blockDim.x) {
        const long long q = t / (3 * per);
        long long r = t - q * 3 * per;
        const int i = (int)(r / per);
        r -= (long long)i * per;
        const int a = (int)(r / ((long long)nk * post));
        r -= (long long)a * nk * post;
        const int k = (int)(r / post), c = (int)(r - (long long)k * post);
        int s = 0;                                       // k = s(s+1)/2 + az with s = ay + az
        while (((s + 1) * (s + 2)) >> 1 <= k) ++s;
        const int az = k - ((s * (s + 1)) >> 1), ay = s - az, ax = l - s;
        const int ei = i == 0 ? ax : i == 1 ? ay : az;
        const int ku = grad_cart_pos(ay + (i == 1), az + (i == 2));
        double v = U[((q * pre + a) * nu + ku) * post + c];
        if (ei > 0) {
            const int kd = grad_cart_pos(ay - (i == 1), az - (i == 2));
            v = fma(-(double)ei, Dn[((q * pre + a) * nd + kd) * post + c], v);
        }
        G[t] = v;
    }
}
// One index of [outer][ncart(l)][inner] -> [outer][2l+1][inner] by the Cartesian->solid matrix of shell l (Eq. 16).
__global__ void __launch_bounds__(256) grad_solid_kernel(const double *__restrict__ in, double *__restrict__ out, long long outer,
                                                         int l, long long inner) {
    __shared__ double C[13 * 28];
    const int nin = ncart(l), nout = nsolid(l);
    for (int i = threadIdx.x; i < nin * nout; i += blockDim.x) C[i] = c_solid[solid_off(l) + i];
    __syncthreads();
    const long long total = outer * nout * inner;
    for (long long t = blockIdx.x * (long long)blockDim.x + threadIdx.x; t < total; t += (long long)gridDim.x * blockDim.x) {
        const long long o = t / (nout * inner);
        const long long r = t - o * nout * inner;
        const int m = (int)(r / inner);
        const long long c = r - m * inner;
        const double *src = in + o * nin * inner + c;
        double s = 0.0;
        for (int k = 0; k < nin; ++k) s = fma(C[m * nin + k], src[k * inner], s);
        out[t] = s;
    }
}

// ket != nullptr: (ab|cd), centres 0..3; X != nullptr: (ab|X), centres 0..2 (the fourth shell is then a one-component dummy);
// W != nullptr (and bra == ket == nullptr): the 2-center (W|X), centres 0 and 2 (dummies in positions 1 and 3).
int md_eri2_impl(const md_shells *X, const md_shells *Y, int64_t npairs, const int32_t *pair_idx, int pure, int layout, double *out,
                 int64_t out_capacity_elems, void *cuda_stream);
int run_grad(const md_pairs *bra, const md_pairs *ket, const md_shells *X, const md_shells *W, long long nq, const int32_t *qidx, int pure,
             int center, double *out, long long cap, cudaStream_t st) {
    if (center < 0 || center > (ket ? 3 : 2) || (W && center == 1) || (pure != 0 && pure != 1) || nq < 0) return MD_EINVAL;
    md_shells dummy{};                                            // l = 0: one component, identity transform
    const md_shells *sh[4] = {W ? W : &bra->a, W ? &dummy : &bra->b, ket ? &ket->a : X, ket ? &ket->b : &dummy};
    const long long nbrap = W ? W->n : bra->npairs, nketp = ket ? ket->npairs : X->n;
    const int l = sh[center]->l;
    if (l + 1 > MD_MAX_L) return MD_EINVAL;                       // the raised shell must be one the kernels serve
    if (!qidx && nq != nbrap * nketp) return MD_EINVAL;
    long long pc = 1, po = 1;                                     // Cartesian / output components of one quartet block
    for (int s = 0; s < 4; ++s) { pc *= ncart(sh[s]->l); po *= ncomp(sh[s]->l, pure); }
    if (3 * po * nq > cap) return MD_ECAPACITY;
    if (nq > 0 && !out) return MD_EINVAL;
    int e = md_init();
    if (e) return e;
    S.last_launches = 0;
    if (nq == 0) return MD_OK;
    int pre = 1, post = 1;
    for (int s = 0; s < center; ++s) pre *= ncart(sh[s]->l);
    for (int s = center + 1; s < 4; ++s) post *= ncart(sh[s]->l);
    const long long perU = pc / ncart(l) * ncart(l + 1), perD = l > 0 ? pc / ncart(l) * ncart(l - 1) : 0, perG = 3 * pc;
    // raised and lowered shell batches: same centres and exponents
    md_pairs pz{};
    md_pairs up[2] = {bra ? *bra : pz, ket ? *ket : pz}, dn[2] = {up[0], up[1]};
    md_shells Xu = X ? *X : dummy, Xd = Xu, Wu = W ? *W : dummy, Wd = Wu;
    md_shells *su = center < 2 ? (W ? &Wu : center == 0 ? &up[0].a : &up[0].b) : !ket ? &Xu : (center == 2 ? &up[1].a : &up[1].b);
    md_shells *sd = center < 2 ? (W ? &Wd : center == 0 ? &dn[0].a : &dn[0].b) : !ket ? &Xd : (center == 2 ? &dn[1].a : &dn[1].b);
    const long long ncoef = (long long)sh[center]->n * sh[center]->K;
    size_t budget = (size_t)64 << 20;
    if (const char *env = getenv("MD_GRAD_CHUNK_BYTES")) budget = (size_t)atoll(env);
    const size_t per_bytes = 8 * (size_t)(perU + perD + (pure ? 2 : 0) * perG);
    const long long chunk = std::max<long long>(1, std::min<long long>(nq, (long long)(budget / std::max<size_t>(per_bytes, 1))));
    double *coefs2 = nullptr, *U = nullptr, *Dn = nullptr, *G0 = nullptr, *G1 = nullptr;
    int32_t *ci = nullptr;
    CK(cudaMallocAsync(&coefs2, (size_t)std::max<long long>(ncoef, 1) * 8, st));
    CK(cudaMallocAsync(&U, (size_t)chunk * (perU + perD) * 8, st));
    Dn = U + chunk * perU;
    if (pure) { CK(cudaMallocAsync(&G0, (size_t)chunk * perG * 16, st)); G1 = G0 + chunk * perG; }
    if (!qidx) CK(cudaMallocAsync(&ci, (size_t)chunk * 2 * sizeof(int32_t), st));
    int launches = 0;
    if (ncoef > 0) { grad_coefs_kernel<<<(unsigned)((ncoef + 255) / 256), 256, 0, st>>>(sh[center]->exps, sh[center]->coefs, coefs2, ncoef); ++launches; }
    su->l = l + 1; su->coefs = coefs2;
    sd->l = l - 1;
    const int ls[4] = {sh[0]->l, sh[1]->l, sh[2]->l, sh[3]->l};
    for (long long q0 = 0; q0 < nq && e == MD_OK; q0 += chunk) {
        const long long m = std::min(chunk, nq - q0);
        const int32_t *qi = qidx ? qidx + 2 * q0 : ci;
        if (!qidx) { product_idx_kernel<<<(unsigned)((m + 255) / 256), 256, 0, st>>>(ci, q0, m, nketp); ++launches; }
        e = W ? md_eri2_impl(&Wu, &Xu, m, qi, 0, MD_LAYOUT_QUARTET_MAJOR, U, m * perU, st)
              : run_call(view(up[0]), ket ? view(up[1]) : view_single(Xu), m, qi, 0, MD_LAYOUT_QUARTET_MAJOR, U, m * perU, st);
        launches += S.last_launches;
        if (e == MD_OK && l > 0) {
            e = W ? md_eri2_impl(&Wd, &Xd, m, qi, 0, MD_LAYOUT_QUARTET_MAJOR, Dn, m * perD, st)
                  : run_call(view(dn[0]), ket ? view(dn[1]) : view_single(Xd), m, qi, 0, MD_LAYOUT_QUARTET_MAJOR, Dn, m * perD, st);
            launches += S.last_launches;
        }
        if (e != MD_OK) break;
        const unsigned grid = (unsigned)std::min<long long>((m * perG + 255) / 256, (long long)S.nsm * 32);
        double *dst = out + q0 * 3 * po;
        grad_combine_kernel<<<grid, 256, 0, st>>>(U, Dn, pure ? G0 : dst, m, l, pre, post);
        ++launches;
        if (pure) {                                               // d, c, b, a in turn; the last pass writes the result
            long long outer = m * 3 * (long long)ncart(ls[0]) * ncart(ls[1]) * ncart(ls[2]), inner = 1;
            double *src = G0, *tmp = G1;
            for (int s = 3; s >= 0; --s) {
                double *to = s == 0 ? dst : tmp;
                const long long total = outer * nsolid(ls[s]) * inner;
                grad_solid_kernel<<<(unsigned)std::min<long long>((total + 255) / 256, (long long)S.nsm * 32), 256, 0, st>>>(src, to, outer, ls[s], inner);
                ++launches;
                inner *= nsolid(ls[s]);
                if (s > 0) outer /= ncart(ls[s - 1]);
                tmp = src; src = to;
            }
        }
    }
    if (ci) cudaFreeAsync(ci, st);
    if (G0) cudaFreeAsync(G0, st);
    cudaFreeAsync(U, st);
    cudaFreeAsync(coefs2, st);
    S.last_launches = launches;
    if (e == MD_OK) CK(cudaGetLastError());
    return e;
}

}  // namespace

extern "C" {

int md_init(void) {
    static std::mutex mu;
    std::lock_guard<std::mutex> lock(mu);
    int dev = 0;
    CK(cudaGetDevice(&dev));
    if (S.init) return S.device == dev ? MD_OK : MD_EINVAL;    // one device per process (include/md_b200.h)
    {   // keep freed scratch in the stream-ordered pool instead of returning it to the driver at every synchronisation
        cudaMemPool_t pool;
        CK(cudaDeviceGetDefaultMemPool(&pool, dev));
        uint64_t keep = ~0ull;
        CK(cudaMemPoolSetAttribute(pool, cudaMemPoolAttrReleaseThreshold, &keep));
    }
    std::vector<uint32_t> herm;
    std::vector<double> solid;
    make_tables(herm, solid);
    CK(upload_tables(herm.data(), solid.data()));
    CK(fused_upload_tables(herm.data(), solid.data()));
    double inv[MD_LTOT + 8];
    inv[0] = 0.0;
    for (int m = 1; m < MD_LTOT + 8; ++m) inv[m] = 1.0 / (2 * m - 1);
    CK(cudaMemcpyToSymbol(c_inv_odd, inv, sizeof(inv)));
    CK(cudaMalloc(&S.boys_tab, sizeof(double) * MD_BOYS_NROW * MD_BOYS_MTAB));
    boys_table_kernel<<<(MD_BOYS_NROW + 63) / 64, 64>>>(S.boys_tab);
    CK(cudaGetLastError());
    CK(cudaDeviceGetAttribute(&S.nsm, cudaDevAttrMultiProcessorCount, dev));
    CK(cudaDeviceGetAttribute(&S.max_smem, cudaDevAttrMaxSharedMemoryPerBlockOptin, dev));
    CK(cudaFuncSetAttribute(eri_generic_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, S.max_smem - 1024));
    CK(cudaFuncSetAttribute(pair_setup_kernel<0>, cudaFuncAttributeMaxDynamicSharedMemorySize, 96 * 1024));
    CK(cudaFuncSetAttribute(pair_setup_kernel<1>, cudaFuncAttributeMaxDynamicSharedMemorySize, 96 * 1024));
    CK(cudaFuncSetAttribute(pair_setup_kernel<2>, cudaFuncAttributeMaxDynamicSharedMemorySize, 96 * 1024));
    CK(cudaFuncSetAttribute(pair_setup_kernel<3>, cudaFuncAttributeMaxDynamicSharedMemorySize, 96 * 1024));
    CK(cudaFuncSetAttribute(pair_setup_kernel<4>, cudaFuncAttributeMaxDynamicSharedMemorySize, 96 * 1024));
    CK(cudaFuncSetAttribute(pair_setup_kernel<5>, cudaFuncAttributeMaxDynamicSharedMemorySize, 96 * 1024));
    CK(cudaFuncSetAttribute(pair_setup_kernel<6>, cudaFuncAttributeMaxDynamicSharedMemorySize, 96 * 1024));
    CK(cudaFuncSetAttribute(eri_warp_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, 112 * 1024));
    CK(fused_init(S.max_smem));
    CK(fused2_init(S.max_smem));
    CK(mma_init(S.max_smem));
    CK(hl_init(S.max_smem, herm.data(), solid.data()));
    CK(lowl_init(S.max_smem));
    CK(eri3s_init(S.max_smem, herm.data(), solid.data()));
    CK(cudaGetSymbolAddress(&S.static_ws, g_static_scratch));   // once per device, with that device current
    CK(cudaDeviceSynchronize());
    S.init = true;
    S.device = dev;
    return MD_OK;
}

// The runtime-l chain on the library's static scratch: no allocation of any kind in this call (include/md_b200.h).
int md_eri4_static(const md_pairs *bra, const md_pairs *ket, int64_t nquartets, const int32_t *quartet_idx, int pure,
                   int layout, double *out, int64_t out_capacity_elems, void *cuda_stream) {
    int e = check_pairs(bra);
    if (e) return e;
    if ((e = check_pairs(ket))) return e;
    if (pure != 0 && pure != 1) return MD_EINVAL;
    if (layout != MD_LAYOUT_QUARTET_MAJOR && layout != MD_LAYOUT_PAPER) return MD_EINVAL;
    if (layout == MD_LAYOUT_PAPER && quartet_idx) return MD_EINVAL;
    const PairView b = view(*bra), k = view(*ket);
    if (nquartets < 0 || (!quartet_idx && nquartets != b.npairs * k.npairs)) return MD_EINVAL;
    const Shape s = shape_of(b, k, pure);
    if ((long long)s.nab * s.ncd * nquartets > out_capacity_elems) return MD_ECAPACITY;
    if (nquartets > 0 && !out) return MD_EINVAL;
    int dev = -1;
    CK(cudaGetDevice(&dev));
    if (!S.init || !S.static_ws || dev != S.device) return MD_ENOTINIT;
    if (generic_ws_bytes(b, k, pure) > MD_STATIC_SCRATCH_BYTES) return MD_ESTATIC;
    S.last_launches = 0;
    if (nquartets == 0) return MD_OK;
    Scratch sc;                                     // not used by the chain once it has its records' address
    return run_generic_once(b, k, nquartets, quartet_idx, pure, layout, out, (cudaStream_t)cuda_stream, true, sc,
                            S.static_ws, nullptr, 0);
}

int64_t md_eri4_static_bytes(const md_pairs *bra, const md_pairs *ket, int pure) {
    int e = check_pairs(bra);
    if (e) return e;
    if ((e = check_pairs(ket))) return e;
    if (pure != 0 && pure != 1) return MD_EINVAL;
    return (int64_t)generic_ws_bytes(view(*bra), view(*ket), pure);
}

int md_eri4(const md_pairs *bra, const md_pairs *ket, int64_t nquartets, const int32_t *quartet_idx, int pure,
            int layout, double *out, int64_t out_capacity_elems, void *cuda_stream) {
    int e = check_pairs(bra);
    if (e) return e;
    if ((e = check_pairs(ket))) return e;
    return run_call(view(*bra), view(*ket), nquartets, quartet_idx, pure, layout, out, out_capacity_elems,
                    (cudaStream_t)cuda_stream);
}

int md_eri3(const md_pairs *bra, const md_shells *X, int64_t ntriplets, const int32_t *triplet_idx, int pure,
            int layout, double *out, int64_t out_capacity_elems, void *cuda_stream) {
    int e = check_pairs(bra);
    if (e) return e;
    if ((e = check_shells(X))) return e;
    return run_call(view(*bra), view_single(*X), ntriplets, triplet_idx, pure, layout, out, out_capacity_elems,
                    (cudaStream_t)cuda_stream);
}

int md_eri4_grad(const md_pairs *bra, const md_pairs *ket, int64_t nquartets, const int32_t *quartet_idx, int pure,
                 int center, double *out, int64_t out_capacity_elems, void *cuda_stream) {
    int e = check_pairs(bra);
    if (e) return e;
    if ((e = check_pairs(ket))) return e;
    return run_grad(bra, ket, nullptr, nullptr, nquartets, quartet_idx, pure, center, out, out_capacity_elems, (cudaStream_t)cuda_stream);
}

int md_eri3_grad(const md_pairs *bra, const md_shells *X, int64_t ntriplets, const int32_t *triplet_idx, int pure, int center,
                 double *out, int64_t out_capacity_elems, void *cuda_stream) {
    int e = check_pairs(bra);
    if (e) return e;
    if ((e = check_shells(X))) return e;
    return run_grad(bra, nullptr, X, nullptr, ntriplets, triplet_idx, pure, center, out, out_capacity_elems, (cudaStream_t)cuda_stream);
}

int md_eri2_grad(const md_shells *X, const md_shells *Y, int64_t npairs, const int32_t *pair_idx, int pure, int center, double *out,
                 int64_t out_capacity_elems, void *cuda_stream) {
    int e = check_shells(X);
    if (e) return e;
    if ((e = check_shells(Y))) return e;
    if (center != 0 && center != 1) return MD_EINVAL;
    return run_grad(nullptr, nullptr, Y, X, npairs, pair_idx, pure, center == 0 ? 0 : 2, out, out_capacity_elems, (cudaStream_t)cuda_stream);
}

int md_exchange(const md_pairs *bra, const md_pairs *ket, int64_t nquartets, const int32_t *quartet_idx, int pure,
                const int32_t *off_a, const int32_t *off_b, const int32_t *off_c, const int32_t *off_d, int64_t nao,
                const double *D, double *K, void *cuda_stream) {
    int e = check_pairs(bra);
    if (e) return e;
    if ((e = check_pairs(ket))) return e;
    if ((pure != 0 && pure != 1) || nquartets < 0 || nao < 0) return MD_EINVAL;
    if (nquartets > 0 && (!off_a || !off_b || !off_c || !off_d || !D || !K)) return MD_EINVAL;
    if ((e = md_init())) return e;
    const int32_t *const off[4] = {off_a, off_b, off_c, off_d};
    return run_exchange(bra, ket, nquartets, quartet_idx, pure, off, nao, D, K, (cudaStream_t)cuda_stream);
}

int md_eri2(const md_shells *X, const md_shells *Y, int64_t npairs, const int32_t *pair_idx, int pure, int layout,
            double *out, int64_t out_capacity_elems, void *cuda_stream) {
    return md_eri2_impl(X, Y, npairs, pair_idx, pure, layout, out, out_capacity_elems, cuda_stream);
}

}  // extern "C"

namespace {
int md_eri2_impl(const md_shells *X, const md_shells *Y, int64_t npairs, const int32_t *pair_idx, int pure, int layout,
                 double *out, int64_t out_capacity_elems, void *cuda_stream) {
    int e = check_shells(X);
    if (e) return e;
    if ((e = check_shells(Y))) return e;
    if (pure != 0 && pure != 1) return MD_EINVAL;
    if (layout != MD_LAYOUT_QUARTET_MAJOR && layout != MD_LAYOUT_PAPER) return MD_EINVAL;
    if (layout == MD_LAYOUT_PAPER && pair_idx) return MD_EINVAL;
    if (npairs < 0 || (!pair_idx && npairs != X->n * Y->n)) return MD_EINVAL;
    if ((long long)ncomp(X->l, pure) * ncomp(Y->l, pure) * npairs > out_capacity_elems) return MD_ECAPACITY;
    if (npairs > 0 && !out) return MD_EINVAL;
    if ((e = md_init())) return e;
    S.last_launches = 0;
    if (npairs == 0) return MD_OK;
    // Both sides are one-centre expansions (Eqs. 6, 8, 11, 12); the runtime-l chain is side-agnostic.
    Scratch sc;
    sc.st = (cudaStream_t)cuda_stream;
    const int saved = S.variant;
    if (S.variant == MD_VARIANT_AUTO || S.variant > MD_VARIANT_WARP || S.variant == MD_VARIANT_FUSED || S.variant == MD_VARIANT_FUSED2)
        S.variant = MD_VARIANT_WARP;                    // warp kernel where the class is small enough, else DMMA
    e = run_generic(view_single(*X), view_single(*Y), npairs, pair_idx, pure, layout, out, sc.st, S.variant != MD_VARIANT_GENERIC, sc);
    S.variant = saved;
    sc.release();
    return e;
}
}  // namespace

extern "C" {

int64_t md_eri4_out_elems(int la, int lb, int lc, int ld, int pure, int64_t n) {
    if (la < 0 || lb < 0 || lc < 0 || ld < 0 || la > MD_MAX_L || lb > MD_MAX_L || lc > MD_MAX_L || ld > MD_MAX_L ||
        n < 0 || (pure != 0 && pure != 1))
        return MD_EINVAL;
    return (int64_t)ncomp(la, pure) * ncomp(lb, pure) * ncomp(lc, pure) * ncomp(ld, pure) * n;
}
int64_t md_eri3_out_elems(int la, int lb, int lX, int pure, int64_t n) {
    return md_eri4_out_elems(la, lb, lX, 0, pure, n);
}

int64_t md_eri4_workspace_bytes(const md_pairs *bra, const md_pairs *ket, int64_t nq, int list_mode, int pure) {
    if (check_pairs(bra) || check_pairs(ket)) return MD_EINVAL;
    return run_query(view(*bra), view(*ket), nq, list_mode, pure);
}
int64_t md_eri3_workspace_bytes(const md_pairs *bra, const md_shells *X, int64_t nt, int list_mode, int pure) {
    if (check_pairs(bra) || check_shells(X)) return MD_EINVAL;
    return run_query(view(*bra), view_single(*X), nt, list_mode, pure);
}

int md_set_workspace(void *p, size_t bytes) {
    S.user_ws = p;
    S.user_bytes = p ? bytes : 0;
    return MD_OK;
}
int md_set_variant(int v) {
    if (v < MD_VARIANT_AUTO || v > MD_VARIANT_ERI3S) return MD_EINVAL;
    S.variant = v;
    return MD_OK;
}
int md_last_variant(void) { return S.last_variant; }
int md_last_launch_count(void) { return S.last_launches; }

int md_boys(int mmax, int scheme, int64_t n, const double *T, double *out, void *cuda_stream) {
    if (mmax < 0 || mmax > MD_LTOT || n < 0 || (n > 0 && (!T || !out)) || scheme < 0 || scheme > 1) return MD_EINVAL;
    int e = md_init();
    if (e) return e;
    if (n == 0) return MD_OK;
    boys_batch_kernel<<<(unsigned)((n + 127) / 128), 128, 0, (cudaStream_t)cuda_stream>>>(mmax, scheme, n, T, S.boys_tab, out);
    CK(cudaGetLastError());
    return MD_OK;
}

int md_fp64_peak(int kind, int seconds_x10, double *tflops, double *ms_out) {
    if (kind < 0 || kind > 3 || !tflops) return MD_EINVAL;
    int e = md_init();
    if (e) return e;
    double *d = nullptr;
    CK(cudaMalloc(&d, 64));
    cudaEvent_t e0, e1;
    CK(cudaEventCreate(&e0));
    CK(cudaEventCreate(&e1));
    // MD_PEAK_SHAPE="blocks_per_sm,threads" (measurement only): occupancy dependence of the issue loops
    int bps = 8, threads = 256;
    if (const char *f = getenv("MD_PEAK_SHAPE")) sscanf(f, "%d,%d", &bps, &threads);
    const int blocks = S.nsm * bps;
    int iters = 4096;
    double flop_per_iter = kind == 0 ? 2.0 * 16 * threads * blocks
                         : kind == 1 ? 512.0 * 8 * (threads / 32) * blocks
                         : kind == 2 ? 2048.0 * 4 * (threads / 32) * blocks
                                     : (2.0 * 64 * 32 + 512.0 * 8) * (threads / 64) * blocks;
    double best = 0, total_ms = 0, ms_best = 0;
    const double budget_ms = 100.0 * (seconds_x10 > 0 ? seconds_x10 : 5);
    for (int rep = 0; rep < 1000 && total_ms < budget_ms; ++rep) {
        CK(cudaEventRecord(e0));
        if (kind == 0) peak_dfma_kernel<<<blocks, threads>>>(d, iters, 0.999999, 1e-9);
        else if (kind == 1) peak_dmma_kernel<<<blocks, threads>>>(d, iters, 0.999999, 1e-9);
        else if (kind == 2) peak_dmma16_kernel<<<blocks, threads>>>(d, iters, 0.999999, 1e-9);
        else peak_mixed_kernel<<<blocks, threads>>>(d, iters, 0.999999, 1e-9);
        CK(cudaEventRecord(e1));
        CK(cudaEventSynchronize(e1));
        float ms = 0;
        CK(cudaEventElapsedTime(&ms, e0, e1));
        total_ms += ms;
        double tf = flop_per_iter * iters / (ms * 1e-3) / 1e12;
        if (rep > 0 && tf > best) { best = tf; ms_best = ms; }
        if (ms < 20) iters *= 2;
    }
    cudaEventDestroy(e0);
    cudaEventDestroy(e1);
    cudaFree(d);
    *tflops = best;
    if (ms_out) *ms_out = ms_best;
    return MD_OK;
}

const char *md_strerror(int code) {
    switch (code) {
        case MD_OK: return "ok";
        case MD_EINVAL: return "invalid argument";
        case MD_ECAPACITY: return "output buffer too small";
        case MD_ECUDA: return "CUDA runtime error";
        case MD_ENOMEM: return "workspace too small";
        case MD_ESTATIC: return "md_eri4_static: pair records exceed MD_STATIC_SCRATCH_BYTES (32 MiB); use md_eri4";
        case MD_ENOTINIT: return "md_eri4_static: call md_init() on this device first";
        default: return "unknown error";
    }
}
const char *md_last_cuda_error(void) { return S.cuda_err; }
int md_version(void) { return 100; }

}  // extern "C"

#include "host_api.inl"
