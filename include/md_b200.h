/*
 * md_b200.h -- C ABI of the B200-native McMurchie-Davidson two-electron integral engine.
 *
 * The library evaluates, in FP64 on one sm_100a GPU, batches of
 *   4-center integrals (ab|cd)   PAPER.md:43-45, Eq. 3
 *   3-center integrals (ab|X)    PAPER.md:39-41, Eq. 2, read as (ab|X) = [X|ab] (reading S5)
 * over contracted Cartesian Gaussian shells (Eqs. 1 and 4) by the
 * McMurchie-Davidson scheme of PAPER.md section II (Eqs. 5-26): primitive-pair Hermite
 * expansion E/H, Boys function, Hermite Coulomb tensor [r]^(0), the two Hermite->AO
 * contractions, and the Cartesian->solid-harmonic transform.  The call shape follows the
 * paper's Listing IV.1: lists of bra and ket shell pairs, a caller-owned
 * target buffer, asynchronous on a CUDA stream.
 *
 * Conventions common to every call
 * --------------------------------
 * Memory.  md_eri4 / md_eri3 take DEVICE pointers for every array (shell data, index lists,
 *   output).  md_eri4_host / md_eri3_host take HOST pointers for every array and perform
 *   the host<->device copies themselves (they synchronise the stream before returning).
 *   The structs themselves are always host memory.  The caller owns every buffer; the
 *   library never frees or reallocates caller memory.  Scratch (per-pair Hermite data,
 *   computed per call and never kept) is taken per call from the CUDA
 *   stream-ordered memory pool on `cuda_stream` and returned to it after the call's last
 *   kernel, unless md_set_workspace gives the library a caller-owned buffer.
 * Asynchrony.  md_eri4 / md_eri3 enqueue work on `cuda_stream` (a cudaStream_t cast to
 *   void*; NULL = the legacy default stream) and return without any synchronisation, as the
 *   paper's compute() does.  Calls in flight on different streams are
 *   independent (each has its own scratch).  With a caller-owned workspace the caller must
 *   order calls that share it (same stream, or events), as for any buffer it owns.
 * Threads and devices.  One device per process: the first call binds the library to the
 *   current device and calls made with another device current return MD_EINVAL.  md_init
 *   is thread-safe; md_set_variant / md_set_workspace / md_last_* are process-wide
 *   measurement and configuration state, so host threads that change them must serialise
 *   their calls.
 * Errors.  Return 0 (MD_OK) or a negative code; nothing is written to `out` on an argument
 *   error.  No exception crosses the ABI.  md_last_cuda_error() returns the CUDA runtime's
 *   text for the most recent MD_ECUDA.
 * Normalisation.  None is applied (the paper states none): a primitive is exactly
 *   PAPER.md Eq. 1 times coefs[k]; every Cartesian component of a shell uses the same coefs.
 * Component order inside a shell of angular momentum l (0 <= l <= MD_MAX_L):
 *   Cartesian (pure = 0): ax = l..0, ay = l-ax..0, az = l-ax-ay  (xx xy xz yy yz zz), (l+1)(l+2)/2.
 *   Solid     (pure = 1): m = -l..+l, Racah-normalised real solid harmonics without
 *     Condon-Shortley phase (S_1,{-1,0,1} = y,z,x; S_20 = zz-(xx+yy)/2), 2l+1 components
 *     (Eqs. 16-17; coefficient formula in DESIGN.md reading O2).
 * Output layouts (n_a.. = component counts, N_ab = n_a n_b, N_cd = n_c n_d):
 *   MD_LAYOUT_QUARTET_MAJOR  out[q*N_ab*N_cd + ((a*n_b + b)*n_c + c)*n_d + d], q = quartet number.
 *   MD_LAYOUT_PAPER          the paper's V[ij,ab,cd,kl], column-major, bra pair ij fastest
 *                            (PAPER.md:198): out[ij + nbra*(ab + N_ab*(cd + N_cd*kl))];
 *                            only for the full bra x ket product (quartet_idx == NULL).
 *   3-center: the same with d absent: [t][a][b][mX].
 */
#ifndef MD_B200_H
#define MD_B200_H

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

#define MD_MAX_L 6            /* s..i */
#define MD_MAX_K 16           /* contraction degree per shell accepted by the engine */

#define MD_OK          0
#define MD_EINVAL    (-1)     /* l outside 0..MD_MAX_L, K outside 1..MD_MAX_K, n < 0, NULL array, bad flag */
#define MD_ECAPACITY (-2)     /* out_capacity_elems smaller than the result */
#define MD_ECUDA     (-3)     /* CUDA runtime error (allocation, launch, copy) */
#define MD_ENOMEM    (-4)     /* caller-set workspace too small for this call */
#define MD_ESTATIC   (-5)     /* md_eri4_static: the call needs more than MD_STATIC_SCRATCH_BYTES of pair records */
#define MD_ENOTINIT  (-6)     /* md_eri4_static: md_init() has not run on the current device (the call never initialises) */

#define MD_LAYOUT_QUARTET_MAJOR 0
#define MD_LAYOUT_PAPER         1

/* Homogeneous shell batch: n shells that share l and K (pairs are grouped by
 * l and contraction degree).  Arrays are row-major. */
typedef struct {
    int32_t l;               /* angular momentum, 0..MD_MAX_L                           */
    int32_t K;               /* contraction degree, 1..MD_MAX_K (Eq. 4)        */
    int64_t n;               /* number of shells                                        */
    const double *center;    /* [n][3]  bohr                                            */
    const double *exps;      /* [n][K]  zeta_k > 0                                      */
    const double *coefs;     /* [n][K]  c_k, already including any normalisation        */
} md_shells;

/* Pair batch: pair i = (a[idx[2i]], b[idx[2i+1]]); idx == NULL means pair i = (a[i], b[i])
 * and then npairs <= min(a.n, b.n).  One (la, lb, Ka, Kb) class per batch. */
typedef struct {
    md_shells a, b;
    int64_t npairs;
    const int32_t *idx;      /* [npairs][2] or NULL */
} md_pairs;

/*
 * (ab|cd) for nquartets quartets (Eq. 3 through Eqs. 7, 19, 21-26).
 *   quartet q = (bra pair quartet_idx[2q], ket pair quartet_idx[2q+1]);
 *   quartet_idx == NULL: the full product, q = ij*ket->npairs + kl, and nquartets must equal
 *   bra->npairs * ket->npairs.
 * Any order of l and K between the four shells is accepted.  Index lists are trusted (no
 * range check on the device).  out must hold md_eri4_out_elems(...) doubles.
 */
int md_eri4(const md_pairs *bra, const md_pairs *ket,
            int64_t nquartets, const int32_t *quartet_idx,
            int pure, int layout,
            double *out, int64_t out_capacity_elems, void *cuda_stream);

/*
 * (ab|X) for ntriplets triplets: the ket is the single shell X expanded about its own
 * centre with the one-centre coefficients of PAPER.md Eqs. 6, 8, 11, 12 (q = zeta_X, Q = X).
 *   triplet t = (bra pair triplet_idx[2t], shell X triplet_idx[2t+1]); NULL = full product,
 *   t = ij*X->n + x.
 */
int md_eri3(const md_pairs *bra, const md_shells *X,
            int64_t ntriplets, const int32_t *triplet_idx,
            int pure, int layout,
            double *out, int64_t out_capacity_elems, void *cuda_stream);

/*
 * 2-center integrals (X|Y) (the metric of density fitting): both sides are single shells
 * expanded about their own centres with the one-centre coefficients of PAPER.md Eqs. 6, 8, 11, 12.
 *   pair t = (X shell pair_idx[2t], Y shell pair_idx[2t+1]); NULL = the full product, t = x*Y->n + y.
 *   out[t][mX][mY] (MD_LAYOUT_QUARTET_MAJOR) or the paper layout with X as the "bra" index.  DEVICE pointers, asynchronous.
 */
int md_eri2(const md_shells *X, const md_shells *Y, int64_t npairs, const int32_t *pair_idx, int pure, int layout,
            double *out, int64_t out_capacity_elems, void *cuda_stream);

/* Host-buffer forms: every array pointer (inside the structs too) is HOST memory.  The call
 * copies inputs to the device, runs the same kernels, copies the result back into `out`
 * and synchronises `cuda_stream` before returning. */
int md_eri4_host(const md_pairs *bra, const md_pairs *ket,
                 int64_t nquartets, const int32_t *quartet_idx,
                 int pure, int layout,
                 double *out, int64_t out_capacity_elems, void *cuda_stream);
int md_eri3_host(const md_pairs *bra, const md_shells *X,
                 int64_t ntriplets, const int32_t *triplet_idx,
                 int pure, int layout,
                 double *out, int64_t out_capacity_elems, void *cuda_stream);

/*
 * Screening, the step before the hot path ("Due to screening these index sets are not Cartesian
 * products"; BASELINE config 5: "All shell quartets passing a Schwarz bound of 1e-12 are evaluated").
 *
 * md_schwarz: Q[i] = sqrt(max over the components ab of |(ab|ab)|) for every pair i of the batch, from the diagonal
 *   integrals of md_eri4 in (i,i) quartet mode (pure selects the component set the maximum runs over).  Q is a DEVICE
 *   array of npairs doubles.  Asynchronous on cuda_stream.
 * md_quartet_list: every (i,j) with Qbra[i]*Qket[j] >= thr (one FP64 multiply), in ascending (i,j) order; same != 0
 *   keeps only j <= i (bra and ket are the same pair list: the unique quartets).  All pointers are DEVICE memory.
 *   *count receives the number of quartets that pass (also when it exceeds capacity); idx receives the first
 *   min(count, capacity) of them as [k][2] = (bra pair, ket pair), ready to be passed to md_eri4 as quartet_idx.
 *   capacity = 0 with idx = NULL only counts.  Asynchronous on cuda_stream.
 */
int md_schwarz(const md_pairs *pairs, int pure, double *Q, void *cuda_stream);
int md_quartet_list(const double *Qbra, int64_t nbra, const double *Qket, int64_t nket, double thr, int same,
                    int32_t *idx, int64_t capacity, int64_t *count, void *cuda_stream);

/*
 * Exchange digestion (Eq. 32; 389-399, Eqs. 33-35): K[b][c] += sum over the listed quartets and the
 * components a, d of (ab|cd) D[a][d], without ever storing the integrals V[ij,ab,cd,kl] of Eq. 33.
 *   bra / ket / quartet_idx / pure as for md_eri4 (4-center only).  off_a..off_d (DEVICE, int32): AO offset of every
 *   shell of the four shell batches (row/column of its first component in D and K).  D and K: DEVICE [nao][nao]
 *   row-major; K is ACCUMULATED into (zero it first); it is the caller's business which quartets it lists (Eq. 32 runs
 *   over all a, d; permutational symmetry is not assumed).
 * Classes with every l <= 2 are digested in the integral kernel's epilogue (one atomic per K row and thread); other
 * classes go through an L2-sized chunk of quartet blocks and a digestion kernel.  Atomic accumulation: the summation
 * order, hence the last bits of K, can differ from run to run.  Asynchronous on cuda_stream.
 */
int md_exchange(const md_pairs *bra, const md_pairs *ket, int64_t nquartets, const int32_t *quartet_idx, int pure,
                const int32_t *off_a, const int32_t *off_b, const int32_t *off_c, const int32_t *off_d, int64_t nao,
                const double *D, double *K, void *cuda_stream);

/*
 * First geometric derivatives of (ab|cd): d/dR_i (ab|cd), R the centre of shell
 * `center` (0, 1, 2, 3 = a, b, c, d), i = x, y, z.  By d/dA_i G_a = 2 zeta G_{a+1_i} - a_i G_{a-1_i} (Eq. 1) the
 * derivative is the Cartesian integral with that shell raised (coefficients 2 zeta_k c_k) minus a_i times the one with
 * it lowered; both come from the integral kernels, the combination and the solid-harmonic transform (Eq. 16) from
 * kernels of their own.  The derivative with respect to the fourth centre follows from the other three (they sum to zero).
 *   bra / ket / quartet_idx / pure / cuda_stream as for md_eri4 (4-center only); the differentiated shell needs
 *   l <= MD_MAX_L - 1 (MD_EINVAL otherwise).
 *   out (DEVICE): [q][i][a][b][c][d], 3 N_ab N_cd doubles per quartet, components as md_eri4 (MD_LAYOUT_QUARTET_MAJOR
 *   only); out_capacity_elems is checked against 3 N_ab N_cd nquartets (MD_ECAPACITY).
 * Scratch (the two Cartesian batches of a chunk of quartets, 64 MiB at most) comes from the stream-ordered pool.
 * Asynchronous on cuda_stream.
 */
int md_eri4_grad(const md_pairs *bra, const md_pairs *ket, int64_t nquartets, const int32_t *quartet_idx, int pure,
                 int center, double *out, int64_t out_capacity_elems, void *cuda_stream);
/* The same for (ab|X): center 0, 1, 2 = a, b, X (the three derivatives sum to zero); out[t][i][a][b][mX], 3 N_ab N_X doubles per
 * triplet; arguments as md_eri3. */
int md_eri3_grad(const md_pairs *bra, const md_shells *X, int64_t ntriplets, const int32_t *triplet_idx, int pure,
                 int center, double *out, int64_t out_capacity_elems, void *cuda_stream);
/* The same for the 2-center (X|Y): center 0 = X, 1 = Y (the two derivatives are opposite); out[t][i][mX][mY]; arguments as md_eri2
 * (MD_LAYOUT_QUARTET_MAJOR). */
int md_eri2_grad(const md_shells *X, const md_shells *Y, int64_t npairs, const int32_t *pair_idx, int pure, int center,
                 double *out, int64_t out_capacity_elems, void *cuda_stream);

/* Number of doubles the result occupies (negative error code on bad arguments). */
int64_t md_eri4_out_elems(int la, int lb, int lc, int ld, int pure, int64_t nquartets);
int64_t md_eri3_out_elems(int la, int lb, int lX, int pure, int64_t ntriplets);

/* Scratch, in bytes, that md_eri4 / md_eri3 would take for exactly this call (same batches,
 * count, list_mode = quartet_idx != NULL, pure) with the kernel variant the library selects
 * for it now (md_set_variant included): per-pair Hermite data (PAPER.md:202
 * "{G, H[ab,p]}[ij,K_b]") or the per-CTA pair tables of the fused kernels; 0 if the kernel
 * needs none.  A buffer of this size given to md_set_workspace is enough for that call.
 * Only the struct fields are read (no device memory).  Negative error code on bad arguments. */
int64_t md_eri4_workspace_bytes(const md_pairs *bra, const md_pairs *ket, int64_t nquartets,
                                int list_mode, int pure);
int64_t md_eri3_workspace_bytes(const md_pairs *bra, const md_shells *X, int64_t ntriplets,
                                int list_mode, int pure);

/* Give the library a caller-owned DEVICE scratch buffer (ptr == NULL returns to the
 * stream-ordered pool).  With a caller buffer a call that needs more returns MD_ENOMEM before
 * anything is launched or written (under MD_VARIANT_AUTO an l <= 2 class first falls back to
 * the fused kernel that needs no scratch). */
int md_set_workspace(void *device_ptr, size_t bytes);

/*
 * md_eri4 for callers that must not allocate (CUDA graph capture, serving loops, harnesses that forbid cudaMalloc):
 * the runtime-l chain (pair setup per side, Eqs. 9-17, then the one-warp-per-quartet, DMMA or DFMA quartet
 * kernel, Eqs. 19-26; what MD_VARIANT_WARP / MD_VARIANT_MMA run) with its per-pair records {G, H[ab,p~]}
 * in a file-scope __device__ array of MD_STATIC_SCRATCH_BYTES inside the library instead of pool scratch.  Same
 * arguments, layouts, result and validation as md_eri4.  The call itself makes no cudaMalloc / cudaMallocAsync / cudaFree
 * and calls no allocating library routine; it only enqueues kernels on cuda_stream.
 *   MD_ENOTINIT  md_init() has not been called in this process (md_init allocates the Boys table; call it once, outside
 *                the region that must not allocate) or another device is current;
 *   MD_ESTATIC   8 * (npairs_bra * Ka*Kb * (4 + N~_bra N_ab) + npairs_ket * Kc*Kd * (4 + N~_ket N_cd)) bytes (each
 *                record rounded to an even number of doubles) exceed MD_STATIC_SCRATCH_BYTES; nothing is launched.
 *                md_eri4_static_bytes() returns that size for a call.
 * The array is one per device and shared by every md_eri4_static call: it keeps the last call's records (each call
 * writes every word it reads, nothing has to start at zero), and two calls that overlap on the GPU (different streams,
 * or two host threads) race on it -- order them on one stream or with events.  Every GPU that loads the library holds
 * the 32 MiB until the process exits.  md_eri4 and the other entry points never touch the array.
 */
#define MD_STATIC_SCRATCH_BYTES ((size_t)32 << 20)
int md_eri4_static(const md_pairs *bra, const md_pairs *ket,
                   int64_t nquartets, const int32_t *quartet_idx, int pure, int layout,
                   double *out, int64_t out_capacity_elems, void *cuda_stream);
/* Bytes of the static array md_eri4_static would use for these batches (struct fields only; negative error code). */
int64_t md_eri4_static_bytes(const md_pairs *bra, const md_pairs *ket, int pure);

/* Kernel-variant control, for measurement:
 *   MD_VARIANT_AUTO    the measured-best variant per class (default)
 *   MD_VARIANT_GENERIC the runtime-l kernel chain (pair setup + DFMA quartet kernel) for every class
 *   MD_VARIANT_FUSED   the compile-time-l fused kernel where one exists, else generic  */
#define MD_VARIANT_AUTO    0
#define MD_VARIANT_GENERIC 1
#define MD_VARIANT_FUSED   2
#define MD_VARIANT_MMA     3     /* pair setup + the DMMA (mma.sync f64) quartet kernel for every class */
#define MD_VARIANT_FUSED2  4     /* the warp-specialised fused kernel where one exists, else as AUTO */
#define MD_VARIANT_WARP    5     /* pair setup + the one-warp-per-quartet kernel where the class is small enough, else as MMA */
#define MD_VARIANT_HL     6     /* the one-launch high-l kernel (in-kernel pair setup, TMA-staged DMMA) where it fits, else as MMA */
#define MD_VARIANT_LOWL   7     /* one thread per quartet, registers only, for classes with every l <= 1 (quartet-major layout), else as AUTO */
#define MD_VARIANT_ERI3S  8     /* one warp per triplet, sparse Cartesian bra, for 3-center classes with la, lb <= 3, else as AUTO */
int md_set_variant(int variant);
/* Which variant the last md_eri4/md_eri3 call used (MD_VARIANT_GENERIC, _FUSED, _MMA, _FUSED2 or _WARP),
 * and how many kernels it launched. */
int md_last_variant(void);
int md_last_launch_count(void);

/* One-time initialisation (Boys table, component tables) on the current device.  Called
 * implicitly by the first compute call; exposed so that timing can exclude it. */
int md_init(void);

/* Boys function F_m(T), m = 0..mmax <= 4*MD_MAX_L, for n values of T (device pointers;
 * out is [n][mmax+1]): the device routines the integral kernels use (Eq. 22).
 *   scheme 0: top order from the Taylor table + downward recursion (runtime-l kernel)
 *   scheme 1: every order from the Taylor table independently (fused kernels) */
int md_boys(int mmax, int scheme, int64_t n, const double *T, double *out, void *cuda_stream);

/* Measurement helper (not on the hot path): best achieved FP64 rate, in TFLOP/s, of a pure
 * issue loop running for about seconds_x10/10 s on the current device.
 *   kind 0: DFMA (vector pipe), 1: DMMA mma.sync.m8n8k4.f64, 2: DMMA mma.sync.m16n8k8.f64,
 *   3: DFMA and DMMA m8n8k4 issued by alternate warps of the same CTA (sum of both flop counts).
 * tflops and ms_out (duration of the best launch; may be NULL) are HOST pointers.  Synchronous. */
int md_fp64_peak(int kind, int seconds_x10, double *tflops, double *ms_out);

const char *md_strerror(int code);
const char *md_last_cuda_error(void);
int md_version(void);

#ifdef __cplusplus
}
#endif
#endif /* MD_B200_H */
