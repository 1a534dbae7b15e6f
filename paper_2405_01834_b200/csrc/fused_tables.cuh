// fused_tables.cuh -- compile-time index and coefficient tables for the fused kernels.
// Everything here is evaluated by the compiler: after full unrolling the kernels contain
// only the non-zero terms, with shared-memory offsets and solid-harmonic coefficients as
// immediates.
#pragma once
#include "common.cuh"

namespace mdb {

// k-th Cartesian component of shell l in the library's order: ax = l..0, ay = l-ax..0.
struct XYZ { int x, y, z; };
__host__ __device__ constexpr XYZ cart_exp(int l, int k) {
    int i = 0;
    for (int x = l; x >= 0; --x)
        for (int y = l - x; y >= 0; --y) {
            if (i == k) return XYZ{x, y, l - x - y};
            ++i;
        }
    return XYZ{0, 0, 0};
}
// k-th (t,u,v) of the degree-sorted Hermite list.
__host__ __device__ constexpr XYZ herm_exp(int k) {
    int n = 0;
    while (nherm(n) <= k) ++n;
    return cart_exp(n, k - nherm(n - 1));
}

__host__ __device__ constexpr double c_sqrt(double x) {
    if (x <= 0) return 0;
    double r = x > 1 ? x : 1;
    for (int i = 0; i < 80; ++i) r = 0.5 * (r + x / r);
    return r;
}
__host__ __device__ constexpr double c_fact(int n) { double r = 1; for (int i = 2; i <= n; ++i) r *= i; return r; }
__host__ __device__ constexpr double c_binom(int n, int k) { return (k < 0 || k > n) ? 0.0 : c_fact(n) / (c_fact(k) * c_fact(n - k)); }

// Cartesian -> Racah-normalised real solid harmonics, C[m+l][cart] (Eqs. 16-17;
// formula: DESIGN.md reading O2).  Compile-time twin of the runtime table in md_b200.cu.
template <int L>
struct SolidTab {
    double c[2 * L + 1][(L + 1) * (L + 2) / 2];
    constexpr SolidTab() : c{} {
        for (int m = -L; m <= L; ++m) {
            const int am = m < 0 ? -m : m, w0 = m < 0 ? 1 : 0;
            double two = 1;
            for (int i = 0; i < am; ++i) two *= 2;
            const double N = c_sqrt(2.0 * c_fact(L + am) * c_fact(L - am) / (m == 0 ? 2.0 : 1.0)) / (two * c_fact(L));
            for (int t = 0; 2 * t + am <= L; ++t) {
                double q = 1;
                for (int i = 0; i < t; ++i) q *= 0.25;
                for (int u = 0; u <= t; ++u)
                    for (int w = w0; w <= am; w += 2) {
                        double v = q * c_binom(L, t) * c_binom(L - t, am + t) * c_binom(t, u) * c_binom(am, w);
                        if ((t + (w - w0) / 2) & 1) v = -v;
                        const int ex = 2 * t + am - 2 * u - w, ey = 2 * u + w;
                        const int k = herm_index(ex, ey, L - ex - ey) - nherm(L - 1);
                        c[m + L][k] += N * v;
                    }
            }
        }
    }
};

// Sparse Hermite expansion of a Cartesian shell pair (l1,l2): the list of non-zero
// E^{t}_{x1 x2} E^{u}_{y1 y2} E^{v}_{z1 z2}, pair component cd = c*ncart(l2)+d major, then
// t, u, v ascending.  off[i] is t*ST + u*SU + v, i.e. the Hermite cube offset (ST = S*S,
// SU = S) for the ket side, or the compact Hermite index when ST = 0 (bra side).
template <int L1, int L2>
struct ProdCount {
    static constexpr int value() {
        int n = 0;
        for (int c = 0; c < ncart(L1); ++c)
            for (int d = 0; d < ncart(L2); ++d) {
                XYZ a = cart_exp(L1, c), b = cart_exp(L2, d);
                n += (a.x + b.x + 1) * (a.y + b.y + 1) * (a.z + b.z + 1);
            }
        return n;
    }
};

template <int L1, int L2, int S>
struct ProdList {
    static constexpr int N = ProdCount<L1, L2>::value();
    short comp[N];
    short off[N];       // S > 0: cube offset; S == 0: compact Hermite index
    constexpr ProdList() : comp{}, off{} {
        int i = 0;
        for (int c = 0; c < ncart(L1); ++c)
            for (int d = 0; d < ncart(L2); ++d) {
                XYZ a = cart_exp(L1, c), b = cart_exp(L2, d);
                for (int t = 0; t <= a.x + b.x; ++t)
                    for (int u = 0; u <= a.y + b.y; ++u)
                        for (int v = 0; v <= a.z + b.z; ++v) {
                            comp[i] = (short)(c * ncart(L2) + d);
                            off[i] = (short)(S > 0 ? (t * S + u) * S + v : herm_index(t, u, v));
                            ++i;
                        }
            }
    }
};

// Runtime twin used by the threads that WRITE the product list: first entry per pair component.
template <int L1, int L2>
struct ProdStart {
    short start[ncart(L1) * ncart(L2) + 1];
    constexpr ProdStart() : start{} {
        int i = 0;
        for (int c = 0; c < ncart(L1); ++c)
            for (int d = 0; d < ncart(L2); ++d) {
                XYZ a = cart_exp(L1, c), b = cart_exp(L2, d);
                start[c * ncart(L2) + d] = (short)i;
                i += (a.x + b.x + 1) * (a.y + b.y + 1) * (a.z + b.z + 1);
            }
        start[ncart(L1) * ncart(L2)] = (short)i;
    }
};
template <int L1, int L2>
__device__ const ProdStart<L1, L2> d_prod_start{};

}  // namespace mdb
