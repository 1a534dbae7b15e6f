// lowl_inst.cu -- instantiations and dispatch of the one-thread-per-quartet kernel (lowl.cuh): all 16 ordered 4-center
// classes and all 8 ordered 3-center classes with every l <= 1 (no canonical swaps: each order has its own instance).
#include <algorithm>

#include "lowl.cuh"
#include "lowl_api.cuh"

namespace mdb {

namespace {
typedef void (*LowlFn)(LowlArgs);
LowlFn g_lowl[2][2][2][2][2];          // [la][lb][lc][ld][single]
int g_lowl_smem[2][2][2][2];
int g_lowl_max_smem = 227 * 1024;

template <int LA, int LB, int LC, int LD>
cudaError_t reg4(int max_smem) {
    g_lowl[LA][LB][LC][LD][0] = lowl_kernel<LA, LB, LC, LD, false>;
    g_lowl_smem[LA][LB][LC][LD] = (2 * LA + 1) * (2 * LB + 1) * (2 * LC + 1) * (2 * LD + 1) * 33 * 8 * (MD_LOWL_THREADS / 32);
    cudaError_t e = cudaFuncSetAttribute(lowl_kernel<LA, LB, LC, LD, false>, cudaFuncAttributeMaxDynamicSharedMemorySize, max_smem);
    if (e != cudaSuccess || LD != 0) return e;
    g_lowl[LA][LB][LC][0][1] = lowl_kernel<LA, LB, LC, 0, true>;
    return cudaFuncSetAttribute(lowl_kernel<LA, LB, LC, 0, true>, cudaFuncAttributeMaxDynamicSharedMemorySize, max_smem);
}
template <int LA, int LB>
cudaError_t reg2(int max_smem) {
    cudaError_t e;
    if ((e = reg4<LA, LB, 0, 0>(max_smem)) != cudaSuccess) return e;
    if ((e = reg4<LA, LB, 0, 1>(max_smem)) != cudaSuccess) return e;
    if ((e = reg4<LA, LB, 1, 0>(max_smem)) != cudaSuccess) return e;
    return reg4<LA, LB, 1, 1>(max_smem);
}
}  // namespace

cudaError_t lowl_init(int max_smem) {
    g_lowl_max_smem = max_smem;
    cudaError_t e;
    if ((e = reg2<0, 0>(max_smem)) != cudaSuccess) return e;
    if ((e = reg2<0, 1>(max_smem)) != cudaSuccess) return e;
    if ((e = reg2<1, 0>(max_smem)) != cudaSuccess) return e;
    return reg2<1, 1>(max_smem);
}

bool lowl_has_class(const PairView &b, const PairView &k) {
    return !b.single && b.a.l <= 1 && b.b.l <= 1 && k.a.l <= 1 && (k.single || k.b.l <= 1);
}

int lowl_dispatch(const PairView &b, const PairView &k, long long nq, const int32_t *qidx, int pure, double *out,
                  const double *boys_tab, int nsm, cudaStream_t st) {
    if (!lowl_has_class(b, k)) return 0;
    const int ld = k.single ? 0 : k.b.l;
    LowlFn fn = g_lowl[b.a.l][b.b.l][k.a.l][ld][k.single ? 1 : 0];
    if (!fn) return 0;
    const int smem = g_lowl_smem[b.a.l][b.b.l][k.a.l][ld];
    LowlArgs g;
    g.bra = b; g.ket = k; g.qidx = qidx; g.nq = nq; g.nket = k.npairs; g.out = out; g.pure = pure; g.boys_tab = boys_tab;
    const int ctas = std::max(1, std::min(8, g_lowl_max_smem / (smem + 1024)));
    const long long nblk = (nq + MD_LOWL_THREADS - 1) / MD_LOWL_THREADS;
    fn<<<(unsigned)std::min<long long>(nblk, (long long)nsm * ctas), MD_LOWL_THREADS, smem, st>>>(g);
    return 1;
}

}  // namespace mdb
