// ge_tail.cuh -- the end piece of a rod whose length does not fit the blocked kernels' vectors.
//
// The temporally blocked 1-D kernels (ge_temporal.cuh, ge_stream.cuh) move 16-byte vectors and want
// nx % V == 0 (V = 2 fp64, 4 fp32); an odd N is nevertheless a first-class case of the scheme (SURVEY.md 8(c)
// "k = 1, N odd": the last node is alone in phase 0 and paired in phase 1).  Instead of falling back to one
// launch per level, ge_run marches the PREFIX of nx' = nx - nx % V nodes with the blocked kernel as if it
// were a rod of its own (its right end then carries a wrong boundary, which spoils at most 2 nodes per level:
// a two-point group reads u_{i-1} .. u_{i+2}) and lets this kernel recompute the end piece:
// one CTA loads the last 4 tb + 4 + nx % V nodes with the true Dirichlet node into shared memory, marches them
// `levels` <= tb levels with the per-level expressions (pair_update_bc: bit-identical), and overwrites the
// last 2 tb + 2 + nx % V nodes of the new level.  Its own left end is a cut: what that spoils (2 nodes per
// level) stays inside the part that is not written.
#pragma once
#include "ge_common.cuh"

namespace ge {

constexpr int kTailThreads = 128;
constexpr int kTailMaxLen = 2048;          // elements of the window (shared memory: 2 x (kTailMaxLen + 1) values)

// w0: first element of the window (even), o0: first element written; both relative to the rod
template <typename T>
__global__ void __launch_bounds__(kTailThreads)
ge1d_tail_kernel(const T* __restrict__ uin, T* __restrict__ uout, int64_t nx, const Coef1<T>* __restrict__ coef,
                 int64_t w0, int64_t o0, int phase0, int levels) {
    __shared__ T buf[2][kTailMaxLen + 2];
    const Coef1<T> k = coef[0];
    const int L = (int)(nx - w0);                 // window elements 0 .. L-1, element L is the Dirichlet node N+1
    for (int j = threadIdx.x; j < L; j += kTailThreads) buf[0][j] = __ldg(uin + w0 + j);
    if (threadIdx.x == 0) { buf[0][L] = k.hi; buf[1][L] = k.hi; }
    __syncthreads();
    int cb = 0;
    for (int lev = 0; lev < levels; ++lev, cb ^= 1) {
        const int ph = (phase0 + lev) & 1;        // w0 is even: left members sit at window elements of parity ph
        const T* __restrict__ x = buf[cb];
        T* __restrict__ y = buf[cb ^ 1];
        if (threadIdx.x == 0 && ph == 1) y[0] = x[0];          // right member of a pair cut by the window (stale)
        for (int j = ph + 2 * threadIdx.x; j < L; j += 2 * kTailThreads) {
            const T a = j > 0 ? x[j - 1] : x[j];
            const T b = x[j], c = x[j + 1];
            const T d = j + 2 <= L ? x[j + 2] : T(0);
            T lo, hi;
            pair_update_bc(a, b, c, d, k, false, j + 1 == L, lo, hi);
            y[j] = lo;
            if (j + 1 < L) y[j + 1] = hi;
        }
        __syncthreads();
    }
    for (int64_t i = o0 + threadIdx.x; i < nx; i += kTailThreads) uout[i] = buf[cb][i - w0];
}

}  // namespace ge
