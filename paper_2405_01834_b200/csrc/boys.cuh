// boys.cuh -- Boys function F_m(T) = int_0^1 y^{2m} exp(-T y^2) dy   (Eq. 22).
//
// The paper says only "interpolation-based"; reading S4 fixes the
// scheme used here:
//   T <  MD_BOYS_TMAX : 8-term Taylor expansion about the nearest grid point T_i = i/16 of a
//                       table of F_m(T_i), m = 0..31, for the TOP order only,
//                         F_M(T_i + h) = sum_k F_{M+k}(T_i) (-h)^k / k!      (dF_m/dT = -F_{m+1})
//                       then the downward recursion F_{m-1} = (2T F_m + e^{-T}) / (2m-1);
//   T >= MD_BOYS_TMAX : F_0 = (1/2) sqrt(pi/T) erf(sqrt T), then the upward recursion
//                         F_{m+1} = ((2m+1) F_m - e^{-T}) / (2T).
// |h| <= 1/32, so the first dropped Taylor term is below (1/32)^8/8! = 2.3e-17 of F_M.
// The fused kernels evaluate each order on its own thread (boys_single): the same Taylor
// expansion for the wanted order m <= 24 (columns m..m+7 <= 31) for T < 128, and
//   F_m(T) = (2m-1)!!/(2T)^m (1/2) sqrt(pi/T)       for T >= 128,
// whose neglected part is below e^{-128} (reading S4) -- no exp, no recursion.
// The table (2049 x 32 doubles, 512 KB) is built on the device at md_init() and stays in L2.
#pragma once
#include "common.cuh"

#define MD_BOYS_MTAB 32
#define MD_BOYS_NROW 2049                 // T_i = i/16, 0 <= T_i <= 128
#define MD_BOYS_TMAX 32.0                 // boys_eval: switch to erf + upward recursion
#define MD_BOYS_TASY 127.96875            // boys_single: switch to the asymptotic form
#define MD_BOYS_STEP 0.0625
#define MD_BOYS_ISTEP 16.0

namespace mdb {

// 1/(2m-1) for the downward recursion (m = 1..24) -- avoids an FP64 division per order.
static __constant__ double c_inv_odd[MD_LTOT + 8];

// Table row i: F_m(i/16), m = 0..31, by the ascending series at m = 31 (all terms positive),
//   F_M(x) = e^{-x} sum_{k>=0} (2x)^k / [(2M+1)(2M+3)..(2M+2k+1)],
// and the downward recursion.  One thread per row; runs once.
static __global__ void boys_table_kernel(double *tab) {
    int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= MD_BOYS_NROW) return;
    const int M = MD_BOYS_MTAB - 1;
    double x = i * MD_BOYS_STEP;
    double term = 1.0 / (2 * M + 1), sum = term;
    for (int k = 1; k < 4000; ++k) {
        term *= 2.0 * x / (2 * M + 2 * k + 1);
        sum += term;
        if (term < 1e-18 * sum) break;
    }
    double ex = exp(-x);
    double f = ex * sum;
    tab[i * MD_BOYS_MTAB + M] = f;
    for (int m = M; m > 0; --m) {
        f = (2.0 * x * f + ex) / (2 * m - 1);
        tab[i * MD_BOYS_MTAB + m - 1] = f;
    }
}

// F[0..mmax] for one T; F may be shared or local memory.  mmax <= 24.
__device__ __forceinline__ void boys_eval(int mmax, double T, const double *__restrict__ tab, double *F) {
    double ex = exp(-T);
    if (T < MD_BOYS_TMAX) {
        int i = __double2int_rn(T * MD_BOYS_ISTEP);
        double mh = i * MD_BOYS_STEP - T;               // -h
        const double *r = tab + i * MD_BOYS_MTAB + mmax;
        double s = r[7] * (1.0 / 5040.0);
        s = fma(s, mh, r[6] * (1.0 / 720.0));
        s = fma(s, mh, r[5] * (1.0 / 120.0));
        s = fma(s, mh, r[4] * (1.0 / 24.0));
        s = fma(s, mh, r[3] * (1.0 / 6.0));
        s = fma(s, mh, r[2] * 0.5);
        s = fma(s, mh, r[1]);
        s = fma(s, mh, r[0]);
        F[mmax] = s;
        double t2 = 2.0 * T;
        for (int m = mmax; m > 0; --m) {
            s = fma(t2, s, ex) * c_inv_odd[m];
            F[m - 1] = s;
        }
    } else {
        double st = sqrt(T);
        double f = 0.88622692545275801365 / st * erf(st);   // sqrt(pi)/2
        double i2t = 0.5 / T;
        F[0] = f;
        for (int m = 0; m < mmax; ++m) {
            f = ((2 * m + 1) * f - ex) * i2t;
            F[m + 1] = f;
        }
    }
}

// One order, independent of the others (fused kernels: one thread per (quartet, m)).
__device__ __forceinline__ double boys_single(int m, double T, const double *__restrict__ tab) {
    if (T < MD_BOYS_TASY) {
        const int i = __double2int_rn(T * MD_BOYS_ISTEP);
        const double mh = i * MD_BOYS_STEP - T;
        const double *r = tab + i * MD_BOYS_MTAB + m;
        double s = __ldg(r + 7) * (1.0 / 5040.0);
        s = fma(s, mh, __ldg(r + 6) * (1.0 / 720.0));
        s = fma(s, mh, __ldg(r + 5) * (1.0 / 120.0));
        s = fma(s, mh, __ldg(r + 4) * (1.0 / 24.0));
        s = fma(s, mh, __ldg(r + 3) * (1.0 / 6.0));
        s = fma(s, mh, __ldg(r + 2) * 0.5);
        s = fma(s, mh, __ldg(r + 1));
        return fma(s, mh, __ldg(r));
    }
    const double it = 1.0 / T;
    double f = 0.88622692545275801365 * sqrt(it);
    const double h = 0.5 * it;
    for (int k = 0; k < m; ++k) f *= (2 * k + 1) * h;
    return f;
}

// Compile-time-order variant: F lives in registers.
template <int M>
__device__ __forceinline__ void boys_eval_t(double T, const double *__restrict__ tab, double (&F)[M + 1]) {
    double ex = exp(-T);
    if (T < MD_BOYS_TMAX) {
        int i = __double2int_rn(T * MD_BOYS_ISTEP);
        double mh = i * MD_BOYS_STEP - T;
        const double *r = tab + i * MD_BOYS_MTAB + M;
        double s = __ldg(r + 7) * (1.0 / 5040.0);
        s = fma(s, mh, __ldg(r + 6) * (1.0 / 720.0));
        s = fma(s, mh, __ldg(r + 5) * (1.0 / 120.0));
        s = fma(s, mh, __ldg(r + 4) * (1.0 / 24.0));
        s = fma(s, mh, __ldg(r + 3) * (1.0 / 6.0));
        s = fma(s, mh, __ldg(r + 2) * 0.5);
        s = fma(s, mh, __ldg(r + 1));
        s = fma(s, mh, __ldg(r + 0));
        F[M] = s;
        double t2 = 2.0 * T;
#pragma unroll
        for (int m = M; m > 0; --m) {
            s = fma(t2, s, ex) * (1.0 / (2 * m - 1));
            F[m - 1] = s;
        }
    } else {
        double st = sqrt(T);
        double f = 0.88622692545275801365 / st * erf(st);
        double i2t = 0.5 / T;
        F[0] = f;
#pragma unroll
        for (int m = 0; m < M; ++m) {
            f = ((2 * m + 1) * f - ex) * i2t;
            F[m + 1] = f;
        }
    }
}

// Test entry (md_boys): out[n][mmax+1].
static __global__ void boys_batch_kernel(int mmax, int scheme, long long n, const double *T, const double *tab, double *out) {
    long long i = blockIdx.x * (long long)blockDim.x + threadIdx.x;
    if (i >= n) return;
    double F[MD_LTOT + 1];
    if (scheme == 0) boys_eval(mmax, T[i], tab, F);
    else for (int m = 0; m <= mmax; ++m) F[m] = boys_single(m, T[i], tab);
    for (int m = 0; m <= mmax; ++m) out[i * (mmax + 1) + m] = F[m];
}

}  // namespace mdb
