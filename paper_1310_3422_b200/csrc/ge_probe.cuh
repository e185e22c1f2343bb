// ge_probe.cuh -- measurement helper, not on the hot path: sustained FFMA / DFMA throughput of the chip.
//
// SURVEY.md 8(d) bounds the temporally blocked and resident kernels by the plain fp32 / fp64 pipes and
// flags the lane counts (128 fp32, 64 fp64 per SM) as an assumption "to be measured with an FMA
// microbenchmark".  This is that microbenchmark: every thread runs CHAINS independent dependent-FMA
// chains (x <- x*a + b), 2048 threads per SM, so latency is covered many times over and the only limit
// left is the issue rate of the pipe at the clock the GPU actually holds.  bench.py times it with CUDA
// events and uses the result as `roofline.peak` of the "alu"-bound kernels.
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

namespace ge {

constexpr int kProbeChains = 8;
constexpr int kProbeUnroll = 32;
constexpr int kProbeThreads = 256;
constexpr int kProbeBlocksPerSm = 8;      // 2048 threads per SM

// DISTINCT: every FMA reads three different registers (x <- x*y[c] + z[c], y and z per chain) instead of sharing its
// multiplier and addend with the other chains -- what the arithmetic of a real kernel looks like to the register
// file: the difference between the two variants is what operand delivery costs on top of the pipe itself.
template <typename T, bool DISTINCT>
__global__ void __launch_bounds__(kProbeThreads, kProbeBlocksPerSm)
ge_fma_probe_kernel(T* __restrict__ sink, T a, T b, int64_t iters) {
    T x[kProbeChains], y[kProbeChains], z[kProbeChains];
#pragma unroll
    for (int c = 0; c < kProbeChains; ++c) {
        x[c] = T(threadIdx.x + c) * a;
        y[c] = DISTINCT ? a - T(c) * T(0.001) : a;
        z[c] = DISTINCT ? b + T(c) * T(0.001) : b;
    }
    // 32 x 8 = 256 FMAs per trip: the counter, compare and branch are 1 % of the issue slots
#pragma unroll 1
    for (int64_t i = 0; i < iters; i += kProbeUnroll) {
#pragma unroll
        for (int u = 0; u < kProbeUnroll; ++u)
#pragma unroll
            for (int c = 0; c < kProbeChains; ++c) x[c] = fma(x[c], y[c], z[c]);
    }
    T s = T(0);
#pragma unroll
    for (int c = 0; c < kProbeChains; ++c) s += x[c];
    // a is chosen < 1 by the host, so the chains converge to b/(1-a): the store below never happens,
    // but the compiler cannot know
    if (s == T(-1)) sink[0] = s;
}

// Enqueues one launch; returns the flops it performs (an FMA counts 2).
template <typename T>
inline cudaError_t fma_probe_launch(T* sink, int64_t iters, int sm_count, double* flops, cudaStream_t s, bool distinct = false) {
    iters = (iters + kProbeUnroll - 1) / kProbeUnroll * kProbeUnroll;
    const int blocks = sm_count * kProbeBlocksPerSm;
    if (distinct) ge_fma_probe_kernel<T, true><<<blocks, kProbeThreads, 0, s>>>(sink, T(0.999), T(0.001), iters);
    else          ge_fma_probe_kernel<T, false><<<blocks, kProbeThreads, 0, s>>>(sink, T(0.999), T(0.001), iters);
    *flops = 2.0 * kProbeChains * (double)iters * (double)blocks * kProbeThreads;
    return cudaGetLastError();
}

}  // namespace ge
