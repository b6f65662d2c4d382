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
