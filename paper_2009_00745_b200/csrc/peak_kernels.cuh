// peak_kernels.cuh -- DFMA-pipe microbenchmark: the measured denominator of the fp64 ("alu") roofline.
// The B200 guides print no fp64 unit count, so bench.py measures it: 16 independent dependent-FMA chains
// per thread, enough warps per SM to saturate the pipe, timed with CUDA events by the caller.
#pragma once
#include "common.cuh"

#define PEAK_CHAINS 16
__global__ void __launch_bounds__(256) k_dfma_peak(double* __restrict__ out, int iters, double a, double b)
{
    double x[PEAK_CHAINS];
#pragma unroll
    for (int i = 0; i < PEAK_CHAINS; ++i) x[i] = 1e-3 * (threadIdx.x + i);
    for (int it = 0; it < iters; ++it) {
#pragma unroll
        for (int i = 0; i < PEAK_CHAINS; ++i) x[i] = fma(x[i], a, b);
    }
    double s = 0.0;
#pragma unroll
    for (int i = 0; i < PEAK_CHAINS; ++i) s += x[i];
    if (s == 123.456) out[blockIdx.x * blockDim.x + threadIdx.x] = s;   // keeps the chains alive
}

// Mixed DMMA / DFMA microbenchmark: per iteration every warp issues NMMA independent m8n8k4 DMMAs and NFMA
// independent DFMAs; answers how the two instruction classes share the fp64 pipe.
template <int NMMA, int NFMA>
__global__ void __launch_bounds__(384) k_fp64_mix(double* __restrict__ out, int iters, double a, double b)
{
    double acc[NMMA > 0 ? NMMA : 1][2];
    double x[NFMA > 0 ? NFMA : 1];
#pragma unroll
    for (int i = 0; i < (NMMA > 0 ? NMMA : 1); ++i) acc[i][0] = acc[i][1] = 1e-3 * (threadIdx.x + i);
#pragma unroll
    for (int i = 0; i < (NFMA > 0 ? NFMA : 1); ++i) x[i] = 1e-3 * (threadIdx.x + i);
    for (int it = 0; it < iters; ++it) {
#pragma unroll
        for (int i = 0; i < (NMMA > NFMA ? NMMA : NFMA); ++i) {
            if (i < NMMA)
                asm volatile("mma.sync.aligned.m8n8k4.row.col.f64.f64.f64.f64 {%0,%1}, {%2}, {%3}, {%0,%1};"
                             : "+d"(acc[i][0]), "+d"(acc[i][1]) : "d"(a), "d"(b));
            if (i < NFMA) x[i] = fma(x[i], a, b);
        }
    }
    double s = 0.0;
#pragma unroll
    for (int i = 0; i < (NMMA > 0 ? NMMA : 1); ++i) s += acc[i][0] + acc[i][1];
#pragma unroll
    for (int i = 0; i < (NFMA > 0 ? NFMA : 1); ++i) s += x[i];
    if (s == 123.456) out[blockIdx.x * blockDim.x + threadIdx.x] = s;
}
