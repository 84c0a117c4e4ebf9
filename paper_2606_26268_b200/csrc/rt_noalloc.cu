// rt_noalloc.cu — rt_cfl_dt_uniform_noalloc: the CFL time step (step 10, L120; R-G15) of a uniform Cartesian grid through
// an entry point that allocates NOTHING: no handle, no cudaMalloc / cudaFree, no allocating library routine.  It is for
// callers that cannot allocate (code under CUDA graph capture, tight serving loops, harnesses that forbid it).
//
// The reduction's scratch is the file-scope device array below, of a fixed size: one slot per x2-x3 row of the grid
// (RT_NOALLOC_MAX_ROWS of them, 512 KB) plus one counter.  Every GPU that loads the library holds it until exit.
// In HOST code the array's name is a host-side stand-in, not a device address: the address the kernel gets comes from
// cudaGetSymbolAddress, looked up once per device with that device current (scratch_of_current_device below).
// All calls share the array: calls that overlap on one GPU (two streams, two threads) race.
#include <cuda_runtime.h>
#include <stdint.h>
#include <stdio.h>
#include <math.h>
#include <mutex>

#include "../../include/rt.h"
#include "rt_kernels_aux.cuh"

namespace rtm1 {

// [0, RT_NOALLOC_MAX_ROWS): bit pattern of each row's maximal rate (rates are >= 0: the unsigned order is the numeric
// order); [RT_NOALLOC_MAX_ROWS]: number of blocks that have finished their rows.  The rest pads to a 256-byte multiple.
static __device__ __align__(256) unsigned long long g_cfl_scratch[RT_NOALLOC_MAX_ROWS + 32];

constexpr int kNaThreads = 256;  // 8 warps; a warp owns one row at a time

struct UniformCfl {
    const double* U[4];
    int n[3];
    int gh[3];
    long long stride1, stride2;  // elements between consecutive x2 / x3 cells of the ghosted arrays
    double il[3];                // 1 / dx_d (0 for an inactive direction: it then adds nothing)
    double chat, cfl;
};

// Same arithmetic per cell as k_cfl (cell_rate_il, rt_kernels_aux.cuh).  Pass 1: every warp writes the maximum of its
// rows into the row's slot.  Pass 2, by the last block to finish: the maximum over the slots, dt = cfl / max.
__global__ void __launch_bounds__(kNaThreads) k_cfl_uniform_noalloc(unsigned long long* __restrict__ scr,
                                                                    const __grid_constant__ UniformCfl a,
                                                                    double* __restrict__ dt_out) {
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    const int nrows = a.n[1] * a.n[2];
    const int wpg = (int)gridDim.x * (kNaThreads / 32);
    for (int row = (int)blockIdx.x * (kNaThreads / 32) + warp; row < nrows; row += wpg) {
        const int j = row % a.n[1], k = row / a.n[1];
        const long long rb = a.gh[0] + (j + a.gh[1]) * a.stride1 + (k + a.gh[2]) * a.stride2;
        double rate = 0.0;
        for (int i = lane; i < a.n[0]; i += 32) {
            const long long id = rb + i;
            rate = dmax(rate, cell_rate_il(a.chat, a.U[0][id], a.U[1][id], a.U[2][id], a.U[3][id], a.il));
        }
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) rate = dmax(rate, __shfl_xor_sync(0xffffffffu, rate, o));
        if (lane == 0) {
            scr[row] = (unsigned long long)__double_as_longlong(rate);
            __threadfence();
        }
    }
    __shared__ bool last;
    __shared__ double sred[kNaThreads / 32];
    __syncthreads();
    if (threadIdx.x == 0) {
        __threadfence();
        const unsigned long long done = atomicAdd(scr + RT_NOALLOC_MAX_ROWS, 1ull);
        last = (done == (unsigned long long)gridDim.x - 1ull);
    }
    __syncthreads();
    if (!last) return;
    __threadfence();
    double v = 0.0;
    for (int row = threadIdx.x; row < nrows; row += kNaThreads) v = dmax(v, __longlong_as_double((long long)__ldcg(scr + row)));
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) v = dmax(v, __shfl_xor_sync(0xffffffffu, v, o));
    if (lane == 0) sred[warp] = v;
    __syncthreads();
    if (threadIdx.x == 0) {
#pragma unroll
        for (int w = 1; w < kNaThreads / 32; ++w) v = dmax(v, sred[w]);
        *dt_out = a.cfl / v;
        scr[RT_NOALLOC_MAX_ROWS] = 0ull;  // re-armed for the next call (the entry point clears it as well)
    }
}

}  // namespace rtm1

using namespace rtm1;

// Device address of g_cfl_scratch on the CURRENT device: cudaGetSymbolAddress once per device, cached.
static cudaError_t scratch_of_current_device(int dev, unsigned long long** out) {
    static std::mutex mtx;
    static unsigned long long* cached[64] = {nullptr};
    std::lock_guard<std::mutex> lk(mtx);
    if (dev >= 0 && dev < 64 && cached[dev]) {
        *out = cached[dev];
        return cudaSuccess;
    }
    unsigned long long* p = nullptr;
    const cudaError_t e = cudaGetSymbolAddress((void**)&p, g_cfl_scratch);
    if (e != cudaSuccess) return e;
    if (dev >= 0 && dev < 64) cached[dev] = p;
    *out = p;
    return cudaSuccess;
}

static int32_t na_fail(char* err, int32_t err_len, int32_t code, const char* msg, const char* detail = nullptr) {
    if (err && err_len > 0) snprintf(err, (size_t)err_len, detail ? "rt_cfl_dt_uniform_noalloc: %s: %s" : "rt_cfl_dt_uniform_noalloc: %s", msg, detail);
    return code;
}

extern "C" int32_t rt_cfl_dt_uniform_noalloc(void* cuda_stream, const int32_t n[3], const double dx[3], double chat, double cfl,
                                             const double* const U[4], double* dt_device, char* err, int32_t err_len) {
    if (err && err_len > 0) err[0] = '\0';
    if (!n || !dx || !U || !dt_device || (reinterpret_cast<uintptr_t>(dt_device) & 7u))
        return na_fail(err, err_len, RT_ERR_INVALID_ARG, "null or misaligned argument");
    if (!(chat > 0.0) || !isfinite(chat) || !(cfl > 0.0) || !isfinite(cfl))
        return na_fail(err, err_len, RT_ERR_INVALID_ARG, "chat and cfl must be finite and > 0");
    bool any_active = false;
    for (int d = 0; d < 3; ++d) {
        if (n[d] < 1) return na_fail(err, err_len, RT_ERR_INVALID_ARG, "n[d] must be >= 1");
        if (n[d] > 1) {
            any_active = true;
            if (!(dx[d] > 0.0) || !isfinite(dx[d])) return na_fail(err, err_len, RT_ERR_INVALID_ARG, "dx[d] of an active direction must be finite and > 0");
        }
    }
    if (!any_active) return na_fail(err, err_len, RT_ERR_INVALID_ARG, "no active direction (every n[d] is 1)");
    const long long nrows = (long long)n[1] * (long long)n[2];
    if (nrows > (long long)RT_NOALLOC_MAX_ROWS) {
        char buf[160];
        snprintf(buf, sizeof(buf), "n[1] * n[2] = %lld x2-x3 rows exceed the static scratch of RT_NOALLOC_MAX_ROWS = %d rows",
                 nrows, (int)RT_NOALLOC_MAX_ROWS);
        return na_fail(err, err_len, RT_ERR_INVALID_ARG, "grid too large", buf);
    }
    for (int q = 0; q < 4; ++q)
        if (!U[q] || (reinterpret_cast<uintptr_t>(U[q]) & 7u)) return na_fail(err, err_len, RT_ERR_INVALID_ARG, "U[q] null or misaligned");

    int dev = -1;
    cudaError_t e = cudaGetDevice(&dev);
    if (e != cudaSuccess) return na_fail(err, err_len, RT_ERR_CUDA, "cudaGetDevice", cudaGetErrorString(e));
    cudaPointerAttributes pa;
    e = cudaPointerGetAttributes(&pa, U[0]);
    if (e != cudaSuccess) {
        cudaGetLastError();
        return na_fail(err, err_len, RT_ERR_INVALID_ARG, "U[0] is not a pointer CUDA knows", cudaGetErrorString(e));
    }
    if (!(pa.type == cudaMemoryTypeManaged || (pa.type == cudaMemoryTypeDevice && pa.device == dev)))
        return na_fail(err, err_len, RT_ERR_INVALID_ARG, "U[0] is not device memory of the CURRENT device (make the fields' device current)");

    unsigned long long* scr = nullptr;
    e = scratch_of_current_device(dev, &scr);
    if (e != cudaSuccess) return na_fail(err, err_len, RT_ERR_CUDA, "cudaGetSymbolAddress(g_cfl_scratch)", cudaGetErrorString(e));

    UniformCfl a;
    long long nt[3];
    for (int d = 0; d < 3; ++d) {
        a.n[d] = n[d];
        a.gh[d] = n[d] > 1 ? 2 : 0;
        nt[d] = (long long)n[d] + 2 * a.gh[d];
        a.il[d] = n[d] > 1 ? 1.0 / dx[d] : 0.0;
    }
    for (int q = 0; q < 4; ++q) a.U[q] = U[q];
    a.stride1 = nt[0];
    a.stride2 = nt[0] * nt[1];
    a.chat = chat;
    a.cfl = cfl;
    cudaStream_t st = reinterpret_cast<cudaStream_t>(cuda_stream);
    // what must start at zero: the blocks-done counter (the row slots are all rewritten before they are read)
    e = cudaMemsetAsync(scr + RT_NOALLOC_MAX_ROWS, 0, sizeof(unsigned long long), st);
    if (e != cudaSuccess) return na_fail(err, err_len, RT_ERR_CUDA, "cudaMemsetAsync", cudaGetErrorString(e));
    const int wpb = kNaThreads / 32;
    long long blocks = (nrows + wpb - 1) / wpb;
    if (blocks > 148 * 8) blocks = 148 * 8;
    k_cfl_uniform_noalloc<<<(unsigned)blocks, kNaThreads, 0, st>>>(scr, a, dt_device);
    e = cudaGetLastError();
    if (e != cudaSuccess) return na_fail(err, err_len, RT_ERR_CUDA, "kernel launch", cudaGetErrorString(e));
    return RT_OK;
}
