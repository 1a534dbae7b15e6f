// peak.cuh -- FP64 peak microbenchmarks (measurement helpers, not part of the hot path).
// MEASURED_PEAKS.json holds no FP64 figure, so bench.py measures the DFMA (vector) and DMMA
// (mma.sync f64) issue rates on the box it runs on and reports them beside the roofline.
#pragma once
#include <cuda_runtime.h>

namespace mdb {

// 16 independent FMA chains per thread; 2*16*iters flop per thread.
__global__ void __launch_bounds__(1024) peak_dfma_kernel(double *out, int iters, double a, double b) {
    double x[16];
#pragma unroll
    for (int i = 0; i < 16; ++i) x[i] = threadIdx.x * 1e-3 + i;
    for (int it = 0; it < iters; ++it) {
#pragma unroll
        for (int i = 0; i < 16; ++i) x[i] = fma(x[i], a, b);
    }
    double s = 0;
#pragma unroll
    for (int i = 0; i < 16; ++i) s += x[i];
    if (s == 12345.678) out[0] = s;            // never true: keeps the chains alive
}

// 8 independent m8n8k4 accumulators per warp; 512 flop per mma per warp.
__global__ void __launch_bounds__(1024) peak_dmma_kernel(double *out, int iters, double a, double b) {
    double c[8][2];
#pragma unroll
    for (int i = 0; i < 8; ++i) { c[i][0] = threadIdx.x * 1e-3; c[i][1] = i; }
    for (int it = 0; it < iters; ++it) {
#pragma unroll
        for (int i = 0; i < 8; ++i)
            asm volatile("mma.sync.aligned.m8n8k4.row.col.f64.f64.f64.f64 {%0,%1}, {%2}, {%3}, {%0,%1};"
                         : "+d"(c[i][0]), "+d"(c[i][1]) : "d"(a), "d"(b));
    }
    double s = 0;
#pragma unroll
    for (int i = 0; i < 8; ++i) s += c[i][0] + c[i][1];
    if (s == 12345.678) out[0] = s;
}

// 4 independent m16n8k8 accumulators per warp (sm_90+ shape); 2*16*8*8 = 2048 flop per mma.
__global__ void __launch_bounds__(1024) peak_dmma16_kernel(double *out, int iters, double a, double b) {
    double c[4][4];
#pragma unroll
    for (int i = 0; i < 4; ++i) { c[i][0] = threadIdx.x * 1e-3; c[i][1] = i; c[i][2] = 1; c[i][3] = 2; }
    for (int it = 0; it < iters; ++it) {
#pragma unroll
        for (int i = 0; i < 4; ++i)
            asm volatile("mma.sync.aligned.m16n8k8.row.col.f64.f64.f64.f64 {%0,%1,%2,%3}, {%4,%5,%6,%7}, {%8,%9}, {%0,%1,%2,%3};"
                         : "+d"(c[i][0]), "+d"(c[i][1]), "+d"(c[i][2]), "+d"(c[i][3])
                         : "d"(a), "d"(b), "d"(a), "d"(b), "d"(a), "d"(b));
    }
    double s = 0;
#pragma unroll
    for (int i = 0; i < 4; ++i) s += c[i][0] + c[i][1] + c[i][2] + c[i][3];
    if (s == 12345.678) out[0] = s;
}

// Mixed: even warps run the DFMA chains, odd warps the m8n8k4 DMMA chains, same iteration count.  If the vector and
// tensor FP64 paths were separate units the sum would exceed either peak; on B200 it does not.
__global__ void __launch_bounds__(1024) peak_mixed_kernel(double *out, int iters, double a, double b) {
    double s = 0;
    if ((threadIdx.x >> 5) & 1) {
        double c[8][2];
#pragma unroll
        for (int i = 0; i < 8; ++i) { c[i][0] = threadIdx.x * 1e-3; c[i][1] = i; }
        for (int it = 0; it < iters; ++it) {
#pragma unroll
            for (int i = 0; i < 8; ++i)
                asm volatile("mma.sync.aligned.m8n8k4.row.col.f64.f64.f64.f64 {%0,%1}, {%2}, {%3}, {%0,%1};"
                             : "+d"(c[i][0]), "+d"(c[i][1]) : "d"(a), "d"(b));
        }
#pragma unroll
        for (int i = 0; i < 8; ++i) s += c[i][0] + c[i][1];
    } else {
        double x[16];
#pragma unroll
        for (int i = 0; i < 16; ++i) x[i] = threadIdx.x * 1e-3 + i;
        for (int it = 0; it < iters; ++it) {            // 64 DFMA = the pipe time of the 8 DMMA above
#pragma unroll
            for (int r = 0; r < 4; ++r)
#pragma unroll
                for (int i = 0; i < 16; ++i) x[i] = fma(x[i], a, b);
        }
#pragma unroll
        for (int i = 0; i < 16; ++i) s += x[i];
    }
    if (s == 12345.678) out[0] = s;
}

}  // namespace mdb
