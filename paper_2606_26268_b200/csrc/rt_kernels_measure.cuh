// rt_kernels_measure.cuh — measurement support, not part of the method: a DFMA microbenchmark that gives bench.py
// the fp64-pipe roof of the device it runs on (SURVEY.md Sect. 8(d): "the build must measure its own fp64 peak
// with a DFMA microbenchmark in the same run").
#pragma once
#include <cuda_runtime.h>

namespace rtm1 {

// Every thread runs CH independent chains of dependent DFMAs, `iters` rounds of 8 per chain.  With enough chains and
// warps the fp64 pipe is the only limit (thread instructions / s = the roof); with CH = 1 and one warp per SM
// sub-partition the time per instruction is the dependent-issue latency of the pipe.
template <int CH, int ROUNDS = 8>
__global__ void __launch_bounds__(1024) k_dfma_chains(double* sink, int iters, double a, double b) {
    double x[CH];
#pragma unroll
    for (int c = 0; c < CH; ++c) x[c] = 1.0 + 1e-3 * (double)(threadIdx.x + c);
#pragma unroll 1
    for (int it = 0; it < iters; ++it) {
#pragma unroll
        for (int r = 0; r < ROUNDS; ++r) {
#pragma unroll
            for (int c = 0; c < CH; ++c) x[c] = fma(x[c], a, b);
        }
    }
    double s = 0.0;
#pragma unroll
    for (int c = 0; c < CH; ++c) s += x[c];
    if (s == 123.456) sink[0] = s;  // never true for the a, b the host passes: keeps the chains alive
}

}  // namespace rtm1
