// screen.cu -- the step BEFORE the hot path ("due to screening these index sets are not
// Cartesian products"): Schwarz factors of a pair batch and the list of shell quartets that pass the bound, on the GPU.
//   Q_ij = sqrt(max_ab |(ab|ab)|)            the diagonal integrals come from md_eri4 in (i,i) quartet mode
//   list = {(i,j): Q_bra[i] Q_ket[j] >= thr}, ascending in (i,j); with same != 0 only j <= i
// Hand-written kernels: iota, diagonal max-abs-sqrt, per-row count (ballot), single-CTA exclusive scan, ordered fill.
#include <algorithm>
#include <cstdint>

#include <cuda_runtime.h>

#include "../../include/md_b200.h"

namespace {

__global__ void iota_pairs_kernel(int32_t *idx, long long n, long long off) {
    const long long i = blockIdx.x * (long long)blockDim.x + threadIdx.x;
    if (i < n) { idx[2 * i] = (int32_t)(off + i); idx[2 * i + 1] = (int32_t)(off + i); }
}

// One warp per pair: max over the diagonal of its [nab][nab] block, then sqrt.
__global__ void diag_max_sqrt_kernel(const double *blk, long long n, int nab, double *Q) {
    const long long w = (blockIdx.x * (long long)blockDim.x + threadIdx.x) >> 5;
    const int lane = threadIdx.x & 31;
    if (w >= n) return;
    const double *b = blk + w * (long long)nab * nab;
    double m = 0.0;
    for (int i = lane; i < nab; i += 32) m = fmax(m, fabs(b[(long long)i * nab + i]));
    for (int o = 16; o; o >>= 1) m = fmax(m, __shfl_xor_sync(0xffffffffu, m, o));
    if (lane == 0) Q[w] = sqrt(m);
}

// Row i of the bound matrix: one CTA; pass 0 counts, pass 1 writes at base[i] + rank in ascending j.
template <int FILL>
__global__ void __launch_bounds__(256) screen_rows_kernel(const double *Qb, long long nb, const double *Qk, long long nk,
                                                          double thr, int same, long long *rowcnt, const long long *base,
                                                          int32_t *idx, long long cap) {
    __shared__ int wsum[8];
    __shared__ long long run;
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    for (long long i = blockIdx.x; i < nb; i += gridDim.x) {
        const double qi = Qb[i];
        const long long jend = same ? min(nk, i + 1) : nk;
        if (threadIdx.x == 0) run = FILL ? base[i] : 0;
        __syncthreads();
        for (long long j0 = 0; j0 < jend; j0 += 256) {
            const long long j = j0 + threadIdx.x;
            const bool keep = j < jend && qi * Qk[j] >= thr;          // one FP64 multiply: the decision the oracle takes
            const unsigned bal = __ballot_sync(0xffffffffu, keep);
            if (lane == 0) wsum[warp] = __popc(bal);
            __syncthreads();
            int before = 0, total = 0;
#pragma unroll
            for (int w = 0; w < 8; ++w) { if (w < warp) before += wsum[w]; total += wsum[w]; }
            if (FILL && keep) {
                const long long pos = run + before + __popc(bal & ((1u << lane) - 1));
                if (pos < cap) { idx[2 * pos] = (int32_t)i; idx[2 * pos + 1] = (int32_t)j; }
            }
            __syncthreads();
            if (threadIdx.x == 0) run += total;
            __syncthreads();
        }
        if (!FILL && threadIdx.x == 0) rowcnt[i] = run;
        __syncthreads();
    }
}

// Exclusive prefix sum of n counts by ONE CTA of 1024 threads (chunked, carry in shared memory); total -> *count.
__global__ void __launch_bounds__(1024) exclusive_scan_kernel(const long long *cnt, long long n, long long *base, long long *count) {
    __shared__ long long wtot[32];
    __shared__ long long carry;
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    if (threadIdx.x == 0) carry = 0;
    __syncthreads();
    for (long long i0 = 0; i0 < n; i0 += 1024) {
        const long long i = i0 + threadIdx.x;
        const long long v = i < n ? cnt[i] : 0;
        long long x = v;
        for (int o = 1; o < 32; o <<= 1) { const long long y = __shfl_up_sync(0xffffffffu, x, o); if (lane >= o) x += y; }
        if (lane == 31) wtot[warp] = x;
        __syncthreads();
        if (warp == 0) {
            long long t = wtot[lane];
            for (int o = 1; o < 32; o <<= 1) { const long long y = __shfl_up_sync(0xffffffffu, t, o); if (lane >= o) t += y; }
            wtot[lane] = t;
        }
        __syncthreads();
        const long long off = carry + (warp ? wtot[warp - 1] : 0);
        if (i < n) base[i] = off + x - v;
        __syncthreads();
        if (threadIdx.x == 0) carry += wtot[31];
        __syncthreads();
    }
    if (threadIdx.x == 0) *count = carry;
}

int ncomp_(int l, int pure) { return pure ? 2 * l + 1 : (l + 1) * (l + 2) / 2; }

}  // namespace

extern "C" {

int md_schwarz(const md_pairs *pairs, int pure, double *Q, void *cuda_stream) {
    if (!pairs || (pure != 0 && pure != 1) || (pairs->npairs > 0 && !Q)) return MD_EINVAL;
    cudaStream_t st = (cudaStream_t)cuda_stream;
    const long long n = pairs->npairs;
    if (n == 0) return MD_OK;
    if (pairs->a.l < 0 || pairs->a.l > MD_MAX_L || pairs->b.l < 0 || pairs->b.l > MD_MAX_L) return MD_EINVAL;
    const int nab = ncomp_(pairs->a.l, pure) * ncomp_(pairs->b.l, pure);
    // (ab|ab) blocks in chunks of at most 256 MB, stream-ordered scratch
    const long long chunk = std::max<long long>(1, std::min<long long>(n, ((long long)256 << 20) / (8LL * nab * nab)));
    double *blk = nullptr;
    int32_t *qi = nullptr;
    if (cudaMallocAsync(&blk, (size_t)chunk * nab * nab * 8, st) != cudaSuccess) return MD_ECUDA;
    if (cudaMallocAsync(&qi, (size_t)chunk * 2 * sizeof(int32_t), st) != cudaSuccess) { cudaFreeAsync(blk, st); return MD_ECUDA; }
    int e = MD_OK;
    for (long long lo = 0; lo < n && e == MD_OK; lo += chunk) {
        const long long m = std::min(chunk, n - lo);
        iota_pairs_kernel<<<(unsigned)((m + 255) / 256), 256, 0, st>>>(qi, m, lo);
        e = md_eri4(pairs, pairs, m, qi, pure, MD_LAYOUT_QUARTET_MAJOR, blk, m * nab * nab, cuda_stream);
        if (e == MD_OK) diag_max_sqrt_kernel<<<(unsigned)((m * 32 + 255) / 256), 256, 0, st>>>(blk, m, nab, Q + lo);
    }
    cudaFreeAsync(qi, st);
    cudaFreeAsync(blk, st);
    if (e == MD_OK && cudaGetLastError() != cudaSuccess) e = MD_ECUDA;
    return e;
}

int md_quartet_list(const double *Qbra, int64_t nbra, const double *Qket, int64_t nket, double thr, int same,
                    int32_t *idx, int64_t capacity, int64_t *count, void *cuda_stream) {
    if (nbra < 0 || nket < 0 || capacity < 0 || !count || (nbra > 0 && !Qbra) || (nket > 0 && !Qket) || (capacity > 0 && !idx) ||
        nbra > 0x7fffffffLL || nket > 0x7fffffffLL)
        return MD_EINVAL;
    cudaStream_t st = (cudaStream_t)cuda_stream;
    if (nbra == 0 || nket == 0) return cudaMemsetAsync(count, 0, sizeof(int64_t), st) == cudaSuccess ? MD_OK : MD_ECUDA;
    long long *rowcnt = nullptr;
    if (cudaMallocAsync(&rowcnt, (size_t)nbra * 2 * sizeof(long long), st) != cudaSuccess) return MD_ECUDA;
    long long *base = rowcnt + nbra;
    const unsigned grid = (unsigned)std::min<long long>(nbra, 148 * 16);
    screen_rows_kernel<0><<<grid, 256, 0, st>>>(Qbra, nbra, Qket, nket, thr, same, rowcnt, nullptr, nullptr, 0);
    exclusive_scan_kernel<<<1, 1024, 0, st>>>(rowcnt, nbra, base, (long long *)count);
    if (capacity > 0) screen_rows_kernel<1><<<grid, 256, 0, st>>>(Qbra, nbra, Qket, nket, thr, same, nullptr, base, idx, capacity);
    cudaFreeAsync(rowcnt, st);
    return cudaGetLastError() == cudaSuccess ? MD_OK : MD_ECUDA;
}

}  // extern "C"
