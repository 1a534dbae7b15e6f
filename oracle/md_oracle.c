/*
 * md_oracle.c -- TEST INFRASTRUCTURE, NOT THE PRODUCT.
 *
 * A plain, slow, double-precision CPU evaluation of the 3-center and 4-center
 * two-electron Coulomb integrals by the textbook McMurchie-Davidson route, written
 * from /root/reference/PAPER.md (arXiv 2405.01834), section II, one shell quartet at a
 * time, with no blocking, batching or fusion.  Only tests/, __graft_entry__.smoke()
 * and bench.py's cpu_baseline / --impl reference legs may call it.  It shares no code,
 * table or constant generator with the CUDA path under paper_2405_01834_b200/csrc/.
 *
 * Every function below cites the passage of PAPER.md it follows.  The readings taken
 * where the paper is silent or garbled are those of SURVEY.md section 8(c) and are
 * listed in DESIGN.md ("Readings of the paper").
 *
 * Parity pins: every function is pinned by tests/test_oracle_*.py (closed forms,
 * identities, an independent Obara-Saika code, library special functions).  Nothing here
 * is "parity unpinned".
 *
 * Build: gcc -O2 -fopenmp -shared -fPIC md_oracle.c -o libmd_oracle.so -lm
 *        add -DORACLE_QUAD -lquadmath for the __float128 build used for roundoff
 *        attribution (same source, same algorithm, wider arithmetic).
 *
 * Conventions:
 *   Cartesian component order inside a shell of angular momentum l:
 *     ax = l..0, ay = l-ax..0, az = l-ax-ay        (xx xy xz yy yz zz for l = 2)
 *   Solid-harmonic component order: m = -l..+l, Racah-normalised real solid harmonics.
 *   Output index: ((a*nb + b)*nc + c)*nd + d, quartet-major.
 *   No normalisation is applied: a primitive is exactly PAPER.md Eq. 1 times c_k.
 */
#include <math.h>
#include <stdint.h>
#include <stdlib.h>
#include <string.h>
#ifdef _OPENMP
#include <omp.h>
#endif

#ifdef ORACLE_QUAD
#include <quadmath.h>
typedef __float128 real;
#define R_EXP expq
#define R_SQRT sqrtq
#define R_ERF erfq
#define R_EPS 1e-36Q
#define R_PI 3.14159265358979323846264338327950288419716939937510Q
#else
typedef double real;
#define R_EXP exp
#define R_SQRT sqrt
#define R_ERF erf
#define R_EPS 1e-17
#define R_PI 3.14159265358979323846264338327950288
#endif

#define LMAX 6              /* per-shell angular momentum limit (s..i)          */
#define LTOT (4 * LMAX)     /* largest Hermite order of [r]^(0): la+lb+lc+ld    */

/* ------------------------------------------------------------------------------------ */
/* Shell component tables                                                               */
/* ------------------------------------------------------------------------------------ */

static int ncart(int l) { return (l + 1) * (l + 2) / 2; }
static int nsolid(int l) { return 2 * l + 1; }

/* Cartesian components (ax,ay,az) of a shell, in the order stated in the header. */
static void cart_list(int l, int (*pw)[3]) {
    int n = 0;
    for (int ax = l; ax >= 0; --ax)
        for (int ay = l - ax; ay >= 0; --ay) {
            pw[n][0] = ax; pw[n][1] = ay; pw[n][2] = l - ax - ay;
            ++n;
        }
}

static real binom(int n, int k) {
    if (k < 0 || k > n) return 0;
    real r = 1;
    for (int i = 1; i <= k; ++i) r = r * (real)(n - k + i) / (real)i;
    return r;
}
static real factorial(int n) { real r = 1; for (int i = 2; i <= n; ++i) r *= i; return r; }

/*
 * Cartesian -> real solid harmonic coefficients C^l_{m,(ax,ay,az)}  (Eqs. 16-17,
 * "C^a_{la ma}", defined by reference to Ref. 31; reading S2/O2 of SURVEY.md 8(c)):
 * the Racah-normalised real solid harmonics in the textbook form of the paper's Ref. 29,
 *   S_lm = N_lm sum_{t=0}^{[(l-|m|)/2]} sum_{u=0}^{t} sum_{v} C^{lm}_{tuv}
 *              x^{2t+|m|-2(u+v)} y^{2(u+v)} z^{l-2t-|m|},
 *   C^{lm}_{tuv} = (-1)^{t+v-v_m} (1/4)^t binom(l,t) binom(l-t,|m|+t) binom(t,u) binom(|m|,2v),
 *   N_lm = 1/(2^{|m|} l!) sqrt(2 (l+|m|)! (l-|m|)! / 2^{delta_m0}),
 *   v = v_m, v_m+1, .., [|m|/2 - v_m] + v_m,  v_m = 0 (m >= 0) or 1/2 (m < 0).
 * Here w = 2v runs over even (m >= 0) or odd (m < 0) integers up to |m|.
 * C is [2l+1][ncart(l)], row index m+l.
 */
static void cart2solid(int l, real *C) {
    int nc = ncart(l);
    int pw[(LMAX + 1) * (LMAX + 2) / 2][3];
    cart_list(l, pw);
    for (int i = 0; i < (2 * l + 1) * nc; ++i) C[i] = 0;
    for (int m = -l; m <= l; ++m) {
        int am = m < 0 ? -m : m;
        real two_am = 1; for (int i = 0; i < am; ++i) two_am *= 2;
        real N = R_SQRT(2 * factorial(l + am) * factorial(l - am) / (m == 0 ? 2 : 1)) / (two_am * factorial(l));
        int w0 = m < 0 ? 1 : 0;
        for (int t = 0; 2 * t <= l - am; ++t) {
            real quarter_t = 1; for (int i = 0; i < t; ++i) quarter_t /= 4;
            for (int u = 0; u <= t; ++u)
                for (int w = w0; w <= am; w += 2) {
                    int sgn_pow = t + (w - w0) / 2;
                    real c = ((sgn_pow & 1) ? -1 : 1) * quarter_t * binom(l, t) * binom(l - t, am + t) * binom(t, u) * binom(am, w);
                    int ex = 2 * t + am - 2 * u - w, ey = 2 * u + w, ez = l - 2 * t - am;
                    for (int k = 0; k < nc; ++k)
                        if (pw[k][0] == ex && pw[k][1] == ey && pw[k][2] == ez) C[(m + l) * nc + k] += N * c;
                }
        }
    }
}

/* ------------------------------------------------------------------------------------ */
/* Boys function  F_m(x) = int_0^1 y^{2m} exp(-x y^2) dy      (Eq. 22)          */
/* ------------------------------------------------------------------------------------ */
/*
 * The paper says only "interpolation-based"; reading O4/S4:
 *   x < 30 : ascending series at the top order M = mmax,
 *              F_M(x) = e^{-x} sum_{i>=0} (2x)^i / [(2M+1)(2M+3)...(2M+2i+1)]   (all terms > 0)
 *            then downward recursion  F_{m-1} = (2x F_m + e^{-x}) / (2m-1).
 *   x >= 30: F_0 = (1/2) sqrt(pi/x) erf(sqrt x), then upward recursion
 *              F_{m+1} = ((2m+1) F_m - e^{-x}) / (2x).
 */
static void boys(int mmax, real x, real *F) {
    real ex = R_EXP(-x);
    if (x < 30) {
        real term = (real)1 / (2 * mmax + 1), sum = term;
        for (int i = 1; i < 2000; ++i) {
            term *= 2 * x / (2 * mmax + 2 * i + 1);
            sum += term;
            if (term < R_EPS * sum) break;
        }
        F[mmax] = ex * sum;
        for (int m = mmax; m > 0; --m) F[m - 1] = (2 * x * F[m] + ex) / (2 * m - 1);
    } else {
        F[0] = R_SQRT(R_PI / x) * R_ERF(R_SQRT(x)) / 2;
        for (int m = 0; m < mmax; ++m) F[m + 1] = ((2 * m + 1) * F[m] - ex) / (2 * x);
    }
}

/* ------------------------------------------------------------------------------------ */
/* Hermite expansion coefficients E                                                     */
/* ------------------------------------------------------------------------------------ */
/*
 * Two-center 1-D table E^t_{ij}, i <= la, j <= lb, t <= la+lb, for one Cartesian axis
 * (Eqs. 9, 10, 13, 14).  xab = A_i - B_i.
 *   seed   E^0_00 = exp(-za zb xab^2 / p)                                   (Eq. 13)
 *   raise i: E^t_{i+1,j} = E^{t-1}_{ij}/(2p) + (P-A) E^t_{ij} + (t+1) E^{t+1}_{ij}   (Eq. 9)
 *   raise j: E^t_{i,j+1} = E^{t-1}_{ij}/(2p) + (P-B) E^t_{ij} + (t+1) E^{t+1}_{ij}   (Eq. 10)
 *   E^t_{ij} = 0 for t outside [0, i+j]                                     (Eq. 14)
 * with P - A = -zb xab / p and P - B = +za xab / p.
 * Layout: E[(i*(lb+1) + j)*(la+lb+1) + t].
 */
static void hermite_E2(int la, int lb, real za, real zb, real xab, real *E) {
    int nt = la + lb + 1;
    real p = za + zb;
    real PA = -zb * xab / p, PB = za * xab / p;
#define E_(i, j, t) E[((i) * (lb + 1) + (j)) * nt + (t)]
    for (int i = 0; i < (la + 1) * (lb + 1) * nt; ++i) E[i] = 0;
    E_(0, 0, 0) = R_EXP(-za * zb * xab * xab / p);
    for (int i = 0; i < la; ++i)          /* Eq. 9 at j = 0 */
        for (int t = 0; t <= i + 1; ++t) {
            real v = PA * E_(i, 0, t);
            if (t > 0) v += E_(i, 0, t - 1) / (2 * p);
            if (t + 1 <= i) v += (t + 1) * E_(i, 0, t + 1);
            E_(i + 1, 0, t) = v;
        }
    for (int i = 0; i <= la; ++i)         /* Eq. 10 */
        for (int j = 0; j < lb; ++j)
            for (int t = 0; t <= i + j + 1; ++t) {
                real v = PB * E_(i, j, t);
                if (t > 0) v += E_(i, j, t - 1) / (2 * p);
                if (t + 1 <= i + j) v += (t + 1) * E_(i, j, t + 1);
                E_(i, j + 1, t) = v;
            }
#undef E_
}

/*
 * One-center 1-D table E^t_a, a <= l, t <= l (Eqs. 8, 11, 12; reading G2):
 *   E^0_0 = 1,  E^t_{a+1} = E^{t-1}_a/(2 za) + (t+1) E^{t+1}_a,  zero outside [0,a] and
 *   for a+t odd.  Stored in the two-center layout with lb = 0: E[a*(l+1) + t].
 */
static void hermite_E1(int l, real za, real *E) {
    int nt = l + 1;
    for (int i = 0; i < (l + 1) * nt; ++i) E[i] = 0;
    E[0] = 1;
    for (int a = 0; a < l; ++a)
        for (int t = 0; t <= a + 1; ++t) {
            real v = 0;
            if (t > 0) v += E[a * nt + t - 1] / (2 * za);
            if (t + 1 <= a) v += (t + 1) * E[a * nt + t + 1];
            E[(a + 1) * nt + t] = v;
        }
}

/* ------------------------------------------------------------------------------------ */
/* Hermite Coulomb tensor  [r]^(m)                                                      */
/* ------------------------------------------------------------------------------------ */
/*
 * PAPER.md Eqs. 21, 23, 24 (readings G5, G6):
 *   [0]^(m) = (-2 rho)^m * 2 pi^{5/2} / (p q sqrt(p+q)) * F_m(rho |P-Q|^2),  rho = p q/(p+q)
 *   [r+1_i]^(m) = r_i [r-1_i]^(m+1) + (P_i - Q_i) [r]^(m+1)
 * R is a dense cube, R[((t*(L+1)) + u)*(L+1) + v] = [tuv]^(0) for t+u+v <= L (other
 * entries are left zero).  W is scratch of (L+2) cubes.
 */
static void hermite_R(int L, real p, real q, const real PQ[3], real *R, real *W) {
    int n1 = L + 1, cube = n1 * n1 * n1;
    real rho = p * q / (p + q);
    real T = rho * (PQ[0] * PQ[0] + PQ[1] * PQ[1] + PQ[2] * PQ[2]);
    real F[LTOT + 1];
    boys(L, T, F);
    real pref = 2 * R_PI * R_PI * R_SQRT(R_PI) / (p * q * R_SQRT(p + q));
#define W_(m, t, u, v) W[(m) * cube + (((t) * n1) + (u)) * n1 + (v)]
    for (int i = 0; i < (L + 1) * cube; ++i) W[i] = 0;
    real pw = 1;
    for (int m = 0; m <= L; ++m) { W_(m, 0, 0, 0) = pw * pref * F[m]; pw *= -2 * rho; }
    for (int m = L - 1; m >= 0; --m)
        for (int t = 0; t <= L - m; ++t)
            for (int u = 0; t + u <= L - m; ++u)
                for (int v = 0; t + u + v <= L - m; ++v) {
                    if (t + u + v == 0) continue;
                    real val;
                    if (t > 0) {
                        val = PQ[0] * W_(m + 1, t - 1, u, v);
                        if (t > 1) val += (t - 1) * W_(m + 1, t - 2, u, v);
                    } else if (u > 0) {
                        val = PQ[1] * W_(m + 1, t, u - 1, v);
                        if (u > 1) val += (u - 1) * W_(m + 1, t, u - 2, v);
                    } else {
                        val = PQ[2] * W_(m + 1, t, u, v - 1);
                        if (v > 1) val += (v - 1) * W_(m + 1, t, u, v - 2);
                    }
                    W_(m, t, u, v) = val;
                }
    for (int i = 0; i < cube; ++i) R[i] = W[i];
#undef W_
}

/* ------------------------------------------------------------------------------------ */
/* One contracted shell quartet, Cartesian components        (Eqs. 3, 4, 7, 19, 25, 26) */
/* ------------------------------------------------------------------------------------ */

typedef struct {
    int l, K;
    const double *center;   /* [3]  */
    const double *exps;     /* [K]  */
    const double *coefs;    /* [K]  */
} shell_t;

/*
 * I[a,b,c,d] += ca cb cc cd * sum_{tuv} E^{ab}_{tuv} sum_{t'u'v'} (-1)^{t'+u'+v'} E^{cd}_{t'u'v'}
 *                                        [t+t', u+u', v+v']^(0)
 * summed over primitives (Eq. 4), in two stages: ket first (Eq. 25), then bra (Eq. 26).
 * one_center_ket != 0 selects the 3-center integral (ab|X): the ket is the single shell
 * c, expanded with the one-center coefficients of Eq. 8 about Q = X with q = zeta_X
 * (reading S5: (ab|X) = [X|ab] of Eq. 2).  Shell d is then ignored (ld = 0).
 * I is [nca][ncb][ncc][ncd] Cartesian, zeroed here.
 */
static void quartet_cart(const shell_t *sa, const shell_t *sb, const shell_t *sc, const shell_t *sd,
                         int one_center_ket, real *I) {
    int la = sa->l, lb = sb->l, lc = sc->l, ld = one_center_ket ? 0 : sd->l;
    int Kd = one_center_ket ? 1 : sd->K;
    int na = ncart(la), nb = ncart(lb), nc = ncart(lc), nd = ncart(ld);
    int Lb = la + lb, Lk = lc + ld, L = Lb + Lk;
    int n1 = L + 1;
    int pa[28][3], pb[28][3], pc[28][3], pd[28][3];
    cart_list(la, pa); cart_list(lb, pb); cart_list(lc, pc); cart_list(ld, pd);

    size_t nout = (size_t)na * nb * nc * nd;
    for (size_t i = 0; i < nout; ++i) I[i] = 0;

    size_t ebra = (size_t)(la + 1) * (lb + 1) * (Lb + 1), eket = (size_t)(lc + 1) * (ld + 1) * (Lk + 1);
    real *Eb = malloc(3 * ebra * sizeof(real)), *Ek = malloc(3 * eket * sizeof(real));
    real *R = malloc((size_t)n1 * n1 * n1 * sizeof(real));
    real *W = malloc((size_t)(L + 1) * n1 * n1 * n1 * sizeof(real));
    int nhb = (Lb + 1) * (Lb + 1) * (Lb + 1);
    real *half = malloc((size_t)nhb * nc * nd * sizeof(real));   /* [p~ | cd] for one primitive quartet */

    for (int ka = 0; ka < sa->K; ++ka)
    for (int kb = 0; kb < sb->K; ++kb) {
        real za = sa->exps[ka], zb = sb->exps[kb], p = za + zb;
        real P[3];
        for (int i = 0; i < 3; ++i) {
            P[i] = (za * sa->center[i] + zb * sb->center[i]) / p;
            hermite_E2(la, lb, za, zb, (real)sa->center[i] - (real)sb->center[i], Eb + i * ebra);
        }
        for (int kc = 0; kc < sc->K; ++kc)
        for (int kd = 0; kd < Kd; ++kd) {
            real zc = sc->exps[kc], q, Q[3], cd_coef;
            if (one_center_ket) {
                q = zc; cd_coef = sc->coefs[kc];
                for (int i = 0; i < 3; ++i) { Q[i] = sc->center[i]; hermite_E1(lc, zc, Ek + i * eket); }
            } else {
                real zd = sd->exps[kd];
                q = zc + zd; cd_coef = (real)sc->coefs[kc] * (real)sd->coefs[kd];
                for (int i = 0; i < 3; ++i) {
                    Q[i] = (zc * sc->center[i] + zd * sd->center[i]) / q;
                    hermite_E2(lc, ld, zc, zd, (real)sc->center[i] - (real)sd->center[i], Ek + i * eket);
                }
            }
            real PQ[3] = {P[0] - Q[0], P[1] - Q[1], P[2] - Q[2]};
            hermite_R(L, p, q, PQ, R, W);
            real coef = (real)sa->coefs[ka] * (real)sb->coefs[kb] * cd_coef;

            /* ket stage, Eq. 25 with Eq. 19: half[tuv][c,d] = sum_{q~} (-1)^{|q~|} E^{cd}_{q~} R_{p~+q~} */
            for (int t = 0; t <= Lb; ++t) for (int u = 0; t + u <= Lb; ++u) for (int v = 0; t + u + v <= Lb; ++v) {
                real *h = half + (size_t)((t * (Lb + 1) + u) * (Lb + 1) + v) * nc * nd;
                for (int c = 0; c < nc; ++c) for (int d = 0; d < nd; ++d) {
                    int cx = pc[c][0], cy = pc[c][1], cz = pc[c][2], dx = pd[d][0], dy = pd[d][1], dz = pd[d][2];
                    const real *ex = Ek + 0 * eket + (size_t)(cx * (ld + 1) + dx) * (Lk + 1);
                    const real *ey = Ek + 1 * eket + (size_t)(cy * (ld + 1) + dy) * (Lk + 1);
                    const real *ez = Ek + 2 * eket + (size_t)(cz * (ld + 1) + dz) * (Lk + 1);
                    real s = 0;
                    for (int t2 = 0; t2 <= cx + dx; ++t2) for (int u2 = 0; u2 <= cy + dy; ++u2) for (int v2 = 0; v2 <= cz + dz; ++v2) {
                        real sign = ((t2 + u2 + v2) & 1) ? -1 : 1;
                        s += sign * ex[t2] * ey[u2] * ez[v2] * R[((t + t2) * n1 + (u + u2)) * n1 + (v + v2)];
                    }
                    h[c * nd + d] = s;
                }
            }
            /* bra stage, Eq. 26: I[ab][cd] += coef * sum_{p~} E^{ab}_{p~} half[p~][cd] */
            for (int a = 0; a < na; ++a) for (int b = 0; b < nb; ++b) {
                int ax = pa[a][0], ay = pa[a][1], az = pa[a][2], bx = pb[b][0], by = pb[b][1], bz = pb[b][2];
                const real *ex = Eb + 0 * ebra + (size_t)(ax * (lb + 1) + bx) * (Lb + 1);
                const real *ey = Eb + 1 * ebra + (size_t)(ay * (lb + 1) + by) * (Lb + 1);
                const real *ez = Eb + 2 * ebra + (size_t)(az * (lb + 1) + bz) * (Lb + 1);
                real *out = I + (size_t)(a * nb + b) * nc * nd;
                for (int t = 0; t <= ax + bx; ++t) for (int u = 0; u <= ay + by; ++u) for (int v = 0; v <= az + bz; ++v) {
                    real e = coef * ex[t] * ey[u] * ez[v];
                    const real *h = half + (size_t)((t * (Lb + 1) + u) * (Lb + 1) + v) * nc * nd;
                    for (int k = 0; k < nc * nd; ++k) out[k] += e * h[k];
                }
            }
        }
    }
    free(Eb); free(Ek); free(R); free(W); free(half);
}

/*
 * Cartesian -> solid transform of one index of a 4-index block (reading O2: applied one
 * index at a time; identical to folding C into H, Eqs. 16-17).
 * in is [n0][ncart(l)][n2], out is [n0][2l+1][n2].
 */
static void solid_index(int l, size_t n0, size_t n2, const real *in, real *out) {
    int nc = ncart(l), ns = nsolid(l);
    real C[(2 * LMAX + 1) * 28];
    cart2solid(l, C);
    for (size_t i0 = 0; i0 < n0; ++i0)
        for (int m = 0; m < ns; ++m)
            for (size_t i2 = 0; i2 < n2; ++i2) {
                real s = 0;
                for (int k = 0; k < nc; ++k) s += C[m * nc + k] * in[(i0 * nc + k) * n2 + i2];
                out[(i0 * ns + m) * n2 + i2] = s;
            }
}

/* One quartet, Cartesian (pure = 0) or solid (pure = 1) output, written as double. */
static void quartet(const shell_t *sa, const shell_t *sb, const shell_t *sc, const shell_t *sd,
                    int one_center_ket, int pure, double *out) {
    int la = sa->l, lb = sb->l, lc = sc->l, ld = one_center_ket ? 0 : sd->l;
    size_t na = ncart(la), nb = ncart(lb), nc = ncart(lc), nd = ncart(ld);
    size_t ncartall = na * nb * nc * nd;
    real *I = malloc(ncartall * sizeof(real)), *T = malloc(ncartall * sizeof(real));
    quartet_cart(sa, sb, sc, sd, one_center_ket, I);
    if (pure) {
        size_t sa_ = nsolid(la), sb_ = nsolid(lb), sc_ = nsolid(lc), sd_ = nsolid(ld);
        solid_index(la, 1, nb * nc * nd, I, T);
        solid_index(lb, sa_, nc * nd, T, I);
        solid_index(lc, sa_ * sb_, nd, I, T);
        solid_index(ld, sa_ * sb_ * sc_, 1, T, I);
        ncartall = sa_ * sb_ * sc_ * sd_;
    }
    for (size_t i = 0; i < ncartall; ++i) out[i] = (double)I[i];
    free(I); free(T);
}

/* ------------------------------------------------------------------------------------ */
/* C entry points (called through ctypes by oracle/__init__.py)                         */
/* ------------------------------------------------------------------------------------ */

int oracle_is_quad(void) {
#ifdef ORACLE_QUAD
    return 1;
#else
    return 0;
#endif
}

int oracle_max_threads(void) {
#ifdef _OPENMP
    return omp_get_max_threads();
#else
    return 1;
#endif
}

void oracle_boys(int mmax, double x, double *F) {
    real f[4 * LTOT + 8];
    boys(mmax, x, f);
    for (int m = 0; m <= mmax; ++m) F[m] = (double)f[m];
}

void oracle_hermite_E2(int la, int lb, double za, double zb, double xab, double *E) {
    int n = (la + 1) * (lb + 1) * (la + lb + 1);
    real *e = malloc(n * sizeof(real));
    hermite_E2(la, lb, za, zb, xab, e);
    for (int i = 0; i < n; ++i) E[i] = (double)e[i];
    free(e);
}

void oracle_hermite_E1(int l, double za, double *E) {
    int n = (l + 1) * (l + 1);
    real *e = malloc(n * sizeof(real));
    hermite_E1(l, za, e);
    for (int i = 0; i < n; ++i) E[i] = (double)e[i];
    free(e);
}

/* R as a dense (L+1)^3 cube, zero where t+u+v > L. */
void oracle_hermite_R(int L, double p, double q, const double *PQ, double *R) {
    int n1 = L + 1, cube = n1 * n1 * n1;
    real *r = malloc(cube * sizeof(real)), *w = malloc((size_t)(L + 1) * cube * sizeof(real));
    real pq[3] = {PQ[0], PQ[1], PQ[2]};
    hermite_R(L, p, q, pq, r, w);
    for (int i = 0; i < cube; ++i) R[i] = (double)r[i];
    free(r); free(w);
}

void oracle_cart2solid(int l, double *C) {
    real c[(2 * LMAX + 1) * 28];
    cart2solid(l, c);
    for (int i = 0; i < (2 * l + 1) * ncart(l); ++i) C[i] = (double)c[i];
}

/*
 * Batch of shell quartets of one class.  Shell batch s (s = a,b,c,d) holds n_s shells of
 * angular momentum l[s] and contraction degree K[s]:
 *   center[s] is [n_s][3], exps[s] is [n_s][K], coefs[s] is [n_s][K].
 * Quartet i uses shells (ia[i], ib[i], ic[i], id[i]).  For three_center != 0 the d batch is
 * ignored and the integral is (ab|X) with X = shell c.  out is quartet-major,
 * out[i*nout + ((a*nb+b)*nc+c)*nd+d].  OpenMP over quartets, nothing else.
 */
void oracle_eri_batch(const int *l, const int *K,
                      const double *const *center, const double *const *exps, const double *const *coefs,
                      int64_t nquartets, const int32_t *ia, const int32_t *ib, const int32_t *ic, const int32_t *id,
                      int three_center, int pure, double *out) {
    int ld = three_center ? 0 : l[3];
    size_t nout = pure ? (size_t)nsolid(l[0]) * nsolid(l[1]) * nsolid(l[2]) * nsolid(ld)
                       : (size_t)ncart(l[0]) * ncart(l[1]) * ncart(l[2]) * ncart(ld);
#pragma omp parallel for schedule(dynamic, 1)
    for (int64_t i = 0; i < nquartets; ++i) {
        shell_t s[4];
        const int32_t idx[4] = {ia[i], ib[i], ic[i], three_center ? 0 : id[i]};
        for (int k = 0; k < (three_center ? 3 : 4); ++k) {
            s[k].l = l[k]; s[k].K = K[k];
            s[k].center = center[k] + 3 * (size_t)idx[k];
            s[k].exps = exps[k] + (size_t)K[k] * idx[k];
            s[k].coefs = coefs[k] + (size_t)K[k] * idx[k];
        }
        if (three_center) s[3] = s[2];
        quartet(&s[0], &s[1], &s[2], &s[3], three_center, pure, out + (size_t)i * nout);
    }
}
