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

// What the issue slot of an SM sub-partition charges for an fp64 instruction: the pipe takes a warp instruction every
// 2 cycles, and the register file delivers one even and one odd 32-bit register per cycle, so a DFMA whose three source
// operands are three different register pairs holds the slot for 3 cycles; one with a constant (or repeated) operand,
// like DMUL and DADD, for 2.  Four independent chains per thread: NREG = 3: x = fma(x, y_c, z_c); NREG = 2:
// x = fma(x, y_c, b) with b a kernel parameter (constant bank).  NF > 0 adds NF independent fp32 multiplies f_j *= g_j
// per group of four DFMAs: they do not hide behind the DFMAs, each takes its own issue cycle.
template <int NREG, int NF>
__global__ void __launch_bounds__(1024) k_dfma_operands(double* sink, int iters, double a, double b, float fa, float fb) {
    constexpr int CH = 4, ROUNDS = 8;
    double x[CH], y[CH], z[CH];
    float f[NF > 0 ? NF : 1], gq[NF > 0 ? NF : 1];
#pragma unroll
    for (int c = 0; c < CH; ++c) {
        x[c] = 1.0 + 1e-3 * (double)(threadIdx.x + c);
        y[c] = a + 1e-12 * (double)(threadIdx.x + c);
        z[c] = b + 1e-12 * (double)(3 * threadIdx.x + c);
    }
#pragma unroll
    for (int j = 0; j < NF; ++j) {
        f[j] = 1.0f + 1e-3f * (float)(threadIdx.x + j);
        gq[j] = fa + fb * (float)(threadIdx.x + j);
    }
#pragma unroll 1
    for (int it = 0; it < iters; ++it) {
#pragma unroll
        for (int r = 0; r < ROUNDS; ++r) {
#pragma unroll
            for (int c = 0; c < CH; ++c) x[c] = NREG == 3 ? fma(x[c], y[c], z[c]) : fma(x[c], y[c], b);
#pragma unroll
            for (int j = 0; j < NF; ++j) f[j] *= gq[j];
        }
    }
    double s = 0.0;
#pragma unroll
    for (int c = 0; c < CH; ++c) s += x[c] + y[c] + z[c];
#pragma unroll
    for (int j = 0; j < NF; ++j) s += (double)f[j] + (double)gq[j];
    if (s == 123.456) sink[0] = s;
}

}  // namespace rtm1
