// fused2_tables.cuh -- compile-time tables of the warp-specialised fused kernel (fused2_kernel.cuh).
#pragma once
#include <utility>

#include "fused_tables.cuh"

namespace mdb {

// static_for<N>(f): f(std::integral_constant<int, I>{}) for I = 0..N-1, so that I is a constant
// expression inside f (register arrays are only ever indexed by constants).
template <class F, int... I>
__device__ __forceinline__ void static_for_impl(F &&f, std::integer_sequence<int, I...>) {
    (f(std::integral_constant<int, I>{}), ...);
}
template <int N, class F>
__device__ __forceinline__ void static_for(F &&f) {
    static_for_impl(static_cast<F &&>(f), std::make_integer_sequence<int, N>{});
}

// Compact 1-D table of one axis: rows (i,j), i <= L1, j <= L2, entries t = 0..i+j (Eq. 14:
// the rest is zero and is not stored).
__host__ __device__ constexpr int e1_rowoff(int L2, int i, int j) {
    int o = 0;
    for (int a = 0; a <= i; ++a)
        for (int b = 0; b <= L2; ++b) {
            if (a == i && b == j) return o;
            o += a + b + 1;
        }
    return o;
}
__host__ __device__ constexpr int e1_count(int L1, int L2) {
    int o = 0;
    for (int a = 0; a <= L1; ++a)
        for (int b = 0; b <= L2; ++b) o += a + b + 1;
    return o;
}

__host__ __device__ constexpr int even_up(int x) { return x + (x & 1); }

// Ket-side sparse Hermite expansion of the Cartesian pair (l1,l2) (Eqs. 7, 14), split into
// NCH chunks of the first shell's components (CHC = ceil(ncart(l1)/NCH) components each) and, inside a
// chunk, ordered q~-major: all products E^{t'}E^{u'}E^{v'} that multiply the same [p~+q~]^(0) are
// adjacent, so the consumer loads that Hermite integral once per q~.
template <int L1, int L2, int NCH>
struct ProdQ {
    static constexpr int NC1 = ncart(L1), NC2 = ncart(L2), NCOMP = NC1 * NC2;
    static constexpr int CHC = (NC1 + NCH - 1) / NCH;
    static constexpr int NH = nherm(L1 + L2);
    static constexpr int N = ProdCount<L1, L2>::value();
    int choff[NCH + 1];          // first list position of each chunk (even), [NCH] = total length
    short start[NCOMP + 1];      // first entry of component cd in (t,u,v)-loop order (producer side)
    short pos[N];                // list position of that entry
    short q_of[N + 2 * NCH];     // per list position: Hermite index q~ (-1 = padding)
    short comp_of[N + 2 * NCH];  // per list position: component inside the chunk, (c - c0)*NC2 + d
    constexpr ProdQ() : choff{}, start{}, pos{}, q_of{}, comp_of{} {
        int i = 0;
        for (int c = 0; c < NC1; ++c)
            for (int d = 0; d < NC2; ++d) {
                XYZ a = cart_exp(L1, c), b = cart_exp(L2, d);
                start[c * NC2 + d] = (short)i;
                i += (a.x + b.x + 1) * (a.y + b.y + 1) * (a.z + b.z + 1);
            }
        start[NCOMP] = (short)i;
        for (int k = 0; k < N + 2 * NCH; ++k) { q_of[k] = -1; comp_of[k] = 0; }
        int w = 0;
        for (int ch = 0; ch < NCH; ++ch) {
            choff[ch] = w;
            const int c0 = ch * CHC, c1 = (c0 + CHC < NC1) ? c0 + CHC : NC1;
            for (int q = 0; q < NH; ++q) {
                XYZ e = herm_exp(q);
                for (int c = c0; c < c1; ++c)
                    for (int d = 0; d < NC2; ++d) {
                        XYZ a = cart_exp(L1, c), b = cart_exp(L2, d);
                        if (e.x > a.x + b.x || e.y > a.y + b.y || e.z > a.z + b.z) continue;
                        // index of (e.x,e.y,e.z) in the component's t,u,v loop nest
                        const int ny = a.y + b.y + 1, nz = a.z + b.z + 1;
                        const int k = (e.x * ny + e.y) * nz + e.z;
                        pos[start[c * NC2 + d] + k] = (short)w;
                        q_of[w] = (short)q;
                        comp_of[w] = (short)((c - c0) * NC2 + d);
                        ++w;
                    }
            }
            w += w & 1;
        }
        choff[NCH] = w;
    }
    constexpr int len() const { return choff[NCH]; }
};
template <int L1, int L2, int NCH>
__device__ const ProdQ<L1, L2, NCH> d_prodq{};

// q~ groups of one chunk of the ProdQ list, for the consumer's software pipeline: group s covers list
// entries [gs[s], gs[s+1]) (relative to the chunk start) and multiplies Hermite index gq[s].
template <int L1, int L2, int NCH, int CH>
struct QGroups {
    static constexpr int NH = nherm(L1 + L2);
    int ng;
    short gs[NH + 1], gq[NH + 1];
    short gid[ProdCount<L1, L2>::value() + 2];      // group of each entry, -1 = padding
    constexpr QGroups() : ng(0), gs{}, gq{}, gid{} {
        constexpr ProdQ<L1, L2, NCH> PQ{};
        const int E0 = PQ.choff[CH], E1 = PQ.choff[CH + 1];
        int last = -2;
        for (int e = E0; e < E1; ++e) {
            const int q = PQ.q_of[e];
            if (q < 0) { gid[e - E0] = -1; continue; }
            if (q != last) { gs[ng] = (short)(e - E0); gq[ng] = (short)q; ++ng; last = q; }
            gid[e - E0] = (short)(ng - 1);
        }
        gs[ng] = (short)(E1 - E0);
    }
};

// Additive ("brick") layout of the Hermite Coulomb tensor [r]^(0), |r| <= L: index(t,u,v) = A t + B u + v.
// It is injective on the simplex t+u+v <= L, so [p~+q~] sits at index(p~) + index(q~) (the Hankel
// structure of PAPER.md Eq. 19 becomes an immediate offset), and (A, B) are chosen (exhaustive search,
// smallest footprint first) so that the bra Hermite rows p~, |p~| <= Lb, fall on the 16 eight-byte
// shared-memory banks with the smallest possible multiplicity: rows that a half-warp reads together are
// then given distinct banks by PMap below.  Rows: {L, Lb, A, B, footprint, max rows per bank}.
struct Brick { int A, B, foot, mult; };
__host__ __device__ constexpr Brick brick_layout(int L, int Lb) {
    constexpr int T[][6] = {
        {0, 0, 1, 1, 1, 1},     {1, 0, 2, 3, 4, 1},     {1, 1, 2, 3, 4, 1},     {2, 0, 4, 6, 13, 1},    {2, 1, 4, 6, 13, 1},
        {2, 2, 4, 6, 13, 1},    {3, 0, 7, 11, 34, 1},   {3, 1, 7, 11, 34, 1},   {3, 2, 10, 14, 43, 1},  {3, 3, 7, 11, 34, 2},
        {4, 0, 11, 15, 61, 1},  {4, 1, 11, 15, 61, 1},  {4, 2, 12, 19, 77, 1},  {4, 3, 11, 18, 73, 2},  {4, 4, 11, 18, 73, 3},
        {5, 0, 16, 22, 111, 1}, {5, 1, 18, 23, 116, 1}, {5, 2, 6, 36, 181, 1},  {5, 3, 18, 23, 116, 2}, {5, 4, 18, 23, 116, 3},
        {6, 0, 22, 28, 169, 1}, {6, 1, 22, 28, 169, 1}, {6, 2, 23, 37, 223, 1}, {6, 3, 22, 35, 211, 2}, {6, 4, 22, 35, 211, 3},
        {7, 0, 29, 37, 260, 1}, {7, 1, 29, 37, 260, 1}, {7, 2, 45, 38, 316, 1}, {7, 3, 40, 29, 281, 2}, {7, 4, 45, 28, 316, 3},
        {8, 0, 45, 37, 361, 1}, {8, 1, 45, 37, 361, 1}, {8, 2, 60, 35, 481, 1}, {8, 3, 50, 39, 401, 2}, {8, 4, 40, 51, 409, 3}};
    for (int i = 0; i < (int)(sizeof(T) / sizeof(T[0])); ++i)
        if (T[i][0] == L && T[i][1] == Lb) return Brick{T[i][2], T[i][3], T[i][4], T[i][5]};
    return Brick{(L + 1) * (L + 1), L + 1, (L + 1) * (L + 1) * (L + 1), 16};      // plain cube
}
__host__ __device__ constexpr bool brick_injective(int L, Brick b) {
    bool seen[1024] = {};
    if (b.foot > 1024) return false;
    int k = 0;
    for (int n = 0; n <= L; ++n)
        for (int t = n; t >= 0; --t)
            for (int u = n - t; u >= 0; --u, ++k) {
                const int i = b.A * t + b.B * u + (n - t - u);
                if (i >= b.foot || seen[i]) return false;
                seen[i] = true;
            }
    return k == nherm(L);
}
// Which Hermite rows each consumer thread owns: slot k of p~ group g holds row p[k][g] (-1 = none).  Rows
// on the same bank (brick index mod 16) go to different slots when the multiplicity allows it, so the PB
// loads a thread issues for one q~ each touch the banks as evenly as the layout permits.
template <int Lb, int PB, int L>
struct PMap {
    static constexpr int NHB = nherm(Lb), NPG = (NHB + PB - 1) / PB;
    short p[PB][NPG];
    constexpr PMap() : p{} {
        if (Lb == 4 && PB == 3 && L == 8) {
            // (dd|dd): rows and lane order found by local search over (A, B, assignment) for the fewest bank
            // conflicts when a half-warp spans two quartets whose buffers are 10 (mod 16) words apart:
            // 13 wavefronts over the 9 distinct half-warp patterns (9 would be conflict-free; the greedy rule gives 18).
            constexpr short T[3][12] = {{10, 0, 18, 28, -1, 19, 21, 7, 26, 24, 16, 30},
                                        {1, 3, 14, 6, 13, 5, 34, 25, 31, 33, 20, 2},
                                        {11, 29, 9, 8, 15, 4, 12, 22, 23, 17, 27, 32}};
            for (int k = 0; k < PB && k < 3; ++k)
                for (int g = 0; g < NPG && g < 12; ++g) p[k][g] = T[k][g];
            return;
        }
        constexpr Brick br = brick_layout(L, Lb);
        int cnt[PB] = {};
        for (int k = 0; k < PB; ++k)
            for (int g = 0; g < NPG; ++g) p[k][g] = -1;
        for (int r = 0; r < 16; ++r) {
            bool used[PB] = {};
            for (int i = 0; i < NHB; ++i) {
                XYZ x = herm_exp(i);
                if ((br.A * x.x + br.B * x.y + x.z) % 16 != r) continue;
                int best = -1;                      // emptiest slot not yet holding this bank, else emptiest slot
                for (int k = 0; k < PB; ++k)
                    if (!used[k] && cnt[k] < NPG && (best < 0 || cnt[k] < cnt[best])) best = k;
                if (best < 0)
                    for (int k = 0; k < PB; ++k)
                        if (cnt[k] < NPG && (best < 0 || cnt[k] < cnt[best])) best = k;
                used[best] = true;
                p[best][cnt[best]++] = (short)i;
            }
        }
    }
};
template <int Lb, int PB, int L>
__device__ const PMap<Lb, PB, L> d_pmap{};

// One word per product-list position: four byte offsets into a table record (fused2_kernel.cuh),
//   byte 0 = the coefficient slot (4: +c_a c_b, 5: -c_a c_b for odd t+u+v, the sign of PAPER.md Eq. 19,
//            6: 0.0 for padding positions), bytes 1-3 = the x, y and z factors (8 + axis*E1 + row + t),
// so that an entry is the product of four shared-memory loads with no select.
__host__ __device__ constexpr unsigned prod_word(int L1, int L2, XYZ a, XYZ b, int t, int u, int v, bool sign) {
    const int E1 = e1_count(L1, L2);
    const unsigned ox = 8 + e1_rowoff(L2, a.x, b.x) + t;
    const unsigned oy = 8 + E1 + e1_rowoff(L2, a.y, b.y) + u;
    const unsigned oz = 8 + 2 * E1 + e1_rowoff(L2, a.z, b.z) + v;
    const unsigned oc = (sign && ((t + u + v) & 1)) ? 5 : 4;
    return oc | ox << 8 | oy << 16 | oz << 24;
}
constexpr unsigned PROD_WORD_ZERO = 6u | 6u << 8 | 6u << 16 | 6u << 24;
// q~-major chunked list (ket side, consumer order of ProdQ).
template <int L1, int L2, int NCH>
struct ProdPackQ {
    static constexpr int LEN = ProdQ<L1, L2, NCH>{}.len();
    unsigned w[LEN];
    constexpr ProdPackQ() : w{} {
        constexpr ProdQ<L1, L2, NCH> PQ{};
        for (int ch = 0; ch < NCH; ++ch)
            for (int e = PQ.choff[ch]; e < PQ.choff[ch + 1]; ++e) {
                if (PQ.q_of[e] < 0) { w[e] = PROD_WORD_ZERO; continue; }
                const int cd = (ch * PQ.CHC) * PQ.NC2 + PQ.comp_of[e];
                XYZ a = cart_exp(L1, cd / PQ.NC2), b = cart_exp(L2, cd % PQ.NC2), h = herm_exp(PQ.q_of[e]);
                w[e] = prod_word(L1, L2, a, b, h.x, h.y, h.z, true);
            }
    }
};
template <int L1, int L2, int NCH>
__device__ const ProdPackQ<L1, L2, NCH> d_packq{};
// component-major list (bra side, order of ProdList), never signed.
template <int L1, int L2>
struct ProdPackC {
    static constexpr int LEN = ProdCount<L1, L2>::value();
    unsigned w[LEN];
    constexpr ProdPackC() : w{} {
        int i = 0;
        for (int c = 0; c < ncart(L1); ++c)
            for (int d = 0; d < ncart(L2); ++d) {
                XYZ a = cart_exp(L1, c), b = cart_exp(L2, d);
                for (int t = 0; t <= a.x + b.x; ++t)
                    for (int u = 0; u <= a.y + b.y; ++u)
                        for (int v = 0; v <= a.z + b.z; ++v) w[i++] = prod_word(L1, L2, a, b, t, u, v, false);
            }
    }
};
template <int L1, int L2>
__device__ const ProdPackC<L1, L2> d_packc{};

// Row offsets of the compact 1-D table, for lane-varying lookups.
template <int L1, int L2>
struct E1Row {
    short off[(L1 + 1) * (L2 + 1)];
    constexpr E1Row() : off{} {
        for (int i = 0; i <= L1; ++i)
            for (int j = 0; j <= L2; ++j) off[i * (L2 + 1) + j] = (short)e1_rowoff(L2, i, j);
    }
};
template <int L1, int L2>
__device__ const E1Row<L1, L2> d_e1row{};

// First N entries of the degree-sorted Hermite list (t | u<<8 | v<<16), for lane-varying lookups.
template <int N>
struct HermTab {
    int e[N];
    constexpr HermTab() : e{} {
        for (int k = 0; k < N; ++k) {
            XYZ a = herm_exp(k);
            e[k] = a.x | (a.y << 8) | (a.z << 16);
        }
    }
};
template <int N>
__device__ const HermTab<N> d_herm{};

// Cartesian -> solid coefficients in device memory, for run-time indexed rows/columns.
template <int L>
__device__ const SolidTab<L> d_solidc{};

// Cartesian exponents of shell l's components, for lane-varying lookups (x | y<<8 | z<<16).
template <int L>
struct CartTab {
    int e[ncart(L)];
    constexpr CartTab() : e{} {
        for (int k = 0; k < ncart(L); ++k) {
            XYZ a = cart_exp(L, k);
            e[k] = a.x | (a.y << 8) | (a.z << 16);
        }
    }
};
template <int L>
__device__ const CartTab<L> d_cart{};

}  // namespace mdb
