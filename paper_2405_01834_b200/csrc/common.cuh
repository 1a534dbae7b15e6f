// common.cuh -- index tables, constants and small helpers shared by every kernel of the engine.
//
// Notation follows PAPER.md section II: la..ld shell angular momenta, Lb = la+lb, Lk = lc+ld,
// L = Lb+Lk; p~ / q~ / r~ Hermite indices (t,u,v); N~(l) = (l+1)(l+2)(l+3)/6 Hermite
// Gaussians of order <= l.
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

#define MD_LMAX 6
#define MD_LTOT (4 * MD_LMAX)
#define MD_NHERM_MAX 2925                       // N~(24)
#define MD_KMAX 16

namespace mdb {

__host__ __device__ constexpr int ncart(int l) { return (l + 1) * (l + 2) / 2; }
__host__ __device__ constexpr int nsolid(int l) { return 2 * l + 1; }
__host__ __device__ constexpr int nherm(int l) { return (l + 1) * (l + 2) * (l + 3) / 6; }
__host__ __device__ constexpr int ncomp(int l, bool pure) { return pure ? nsolid(l) : ncart(l); }

// Offset of the Cartesian->solid matrix of shell l inside c_solid ([2l+1][ncart(l)] each).
__host__ __device__ constexpr int solid_off(int l) {
    int o = 0;
    for (int k = 0; k < l; ++k) o += nsolid(k) * ncart(k);
    return o;
}
#define MD_SOLID_TOTAL 840                      // solid_off(7)

// Degree-sorted list of (t,u,v): all triples of total degree 0, then 1, ..; inside a degree
// n the order is t = n..0, u = n-t..0, v = n-t-u.  Consequences used throughout:
//  * the triples of degree <= n are the first N~(n) entries (one table serves every L);
//  * the Cartesian components of a shell l, in the library's component order
//    (include/md_b200.h), are entries N~(l-1) .. N~(l)-1.
// Packed as t | u<<8 | v<<16 | n<<24.
static __constant__ uint32_t c_herm[MD_NHERM_MAX];
// Cartesian -> real solid harmonic coefficients (Eqs. 16-17), all l <= 6.
static __constant__ double c_solid[MD_SOLID_TOTAL];
// Every translation unit that uses the tables holds its own copy and uploads it with this.
static inline cudaError_t upload_tables(const uint32_t *herm, const double *solid) {
    cudaError_t e = cudaMemcpyToSymbol(c_herm, herm, sizeof(uint32_t) * MD_NHERM_MAX);
    if (e != cudaSuccess) return e;
    return cudaMemcpyToSymbol(c_solid, solid, sizeof(double) * MD_SOLID_TOTAL);
}

__device__ __forceinline__ void unpack_tuv(uint32_t w, int &t, int &u, int &v) {
    t = w & 0xff; u = (w >> 8) & 0xff; v = (w >> 16) & 0xff;
}

// Position of (t,u,v) in the degree-sorted list.
__host__ __device__ constexpr int herm_index(int t, int u, int v) {
    int n = t + u + v;
    return n * (n + 1) * (n + 2) / 6 + (n - t) * (n - t + 1) / 2 + (n - t - u);
}

// Device views of the caller's shell and pair batches (include/md_b200.h).
struct ShellView {
    const double *center, *exps, *coefs;
    int l, K;
};
struct PairView {
    ShellView a, b;
    const int32_t *idx;        // [npairs][2] or nullptr
    long long npairs;
    int single;                // 1: one-centre "pair" (3-center X): shell b is absent
};

// ---- S1: one Cartesian axis of the two-centre Hermite expansion, by one warp (lane = t) -----------------------------
//   E^0_00 = exp(-za zb xab^2/p)                                              (Eq. 13)
//   E^t_{i,j+1} = E^{t-1}_{ij}/(2p) + (P-B) E^t_{ij} + (t+1) E^{t+1}_{ij}     (Eq. 10), along i = 0
//   E^t_{i+1,j} = E^{t-1}_{ij}/(2p) + (P-A) E^t_{ij} + (t+1) E^{t+1}_{ij}     (Eq. 9),  for every j
// E[(i*(lb+1)+j)*nt + t], nt = la+lb+1 <= 13; entries with t > i+j are written as exact zeros (Eq. 14), which the
// H build relies on.  A one-centre expansion (Eq. 8) is the case zb = 0, xab = 0.
__device__ __forceinline__ void hl_e_axis_warp(int la, int lb, double za, double zb, double xab, double *E, int lane) {
    const int nt = la + lb + 1;
    const double p = za + zb, h = 0.5 / p;
    const double xpa = -zb * xab / p, xpb = za * xab / p;
    const double tp1 = (double)(lane + 1);
    double e = lane == 0 ? exp(-za * zb / p * xab * xab) : 0.0;
    if (lane < nt) E[lane] = e;
    for (int j = 0; j < lb; ++j) {
        double em = __shfl_up_sync(0xffffffffu, e, 1), ep = __shfl_down_sync(0xffffffffu, e, 1);
        if (lane == 0) em = 0.0;
        if (lane == 31) ep = 0.0;
        e = xpb * e + h * em + tp1 * ep;
        if (lane < nt) E[(j + 1) * nt + lane] = e;
    }
    for (int j = 0; j <= lb; ++j) {
        e = lane < nt ? E[j * nt + lane] : 0.0;
        for (int i = 0; i < la; ++i) {
            double em = __shfl_up_sync(0xffffffffu, e, 1), ep = __shfl_down_sync(0xffffffffu, e, 1);
            if (lane == 0) em = 0.0;
            if (lane == 31) ep = 0.0;
            e = xpa * e + h * em + tp1 * ep;
            if (lane < nt) E[((i + 1) * (lb + 1) + j) * nt + lane] = e;
        }
    }
}


}  // namespace mdb
