// ge_level_src.cuh -- strategy A (1-D, two-point groups) with non-constant problem
// data (reading R-N3): a source term and
// time-dependent boundary values,  u_t = u_xx + f(x,t),  u(0,t) = lo(t),  u(1,t) = hi(t).
// The paper's model problem has neither; PAPER.md:37 names the
// diffusion step inside an operator splitting as the use.
//
// Saul'yev's asymmetric equations gain s_i = tau f_i at their node, so the pair's
// right-hand sides become p = old_i + r (old_{i-1} - old_i) + s_i and
// q = old_{i+1} + r (old_{i+2} - old_{i+1}) + s_{i+1}; the 2x2 solve is unchanged
// (w = g (q - p), new_i = p + w, new_{i+1} = q - w).  A boundary node read at the
// old level contributes its OLD value, the new-level neighbour of a truncated
// pair its NEW value:  node 1 alone: new = q - e (q - lo_new);  node N alone:
// new = p + e (hi_new - p).
//
// One thread per pair (phase 0: elements (0,1),(2,3),...; phase 1: element 0
// alone, then (1,2),...); the four old values and the two source values come
// through L1, HBM sees every line once: 3 * sizeof(T) algorithmic bytes per
// update (u in, s in, u out).
#pragma once
#include "ge_common.cuh"

namespace ge {

template <typename T>
struct SrcBc { T lo_old, lo_new, hi_old, hi_new; };

constexpr int kSrcThreads = 256;

template <typename T, int PH>
__global__ void __launch_bounds__(kSrcThreads)
ge1d_level_src_kernel(const T* __restrict__ uin, T* __restrict__ uout, const T* __restrict__ src, int64_t nx,
                      const Coef1<T>* __restrict__ coef, const SrcBc<T> bc) {
    const int64_t m = (int64_t)blockIdx.x * kSrcThreads + threadIdx.x;
    const int64_t e = 2 * m - PH;                 // element of the pair's left member (-1: node 0)
    if (e >= nx) return;
    const Coef1<T> k = coef[0];
    auto old = [&](int64_t i) -> T {              // element i of the old level, boundaries at -1 and nx
        if (i < 0) return bc.lo_old;
        if (i >= nx) return bc.hi_old;
        return __ldg(uin + i);
    };
    auto s = [&](int64_t i) -> T { return (src && i >= 0 && i < nx) ? __ldg(src + i) : T(0); };
    const T a = old(e - 1), b = old(e), c = old(e + 1), d = old(e + 2);
    T p = fma(k.r, a - b, b) + s(e);
    T q = fma(k.r, d - c, c) + s(e + 1);
    T g = k.g;
    if (e < 0) { p = bc.lo_new; g = k.e; }        // left member is node 0
    if (e + 1 >= nx) { q = bc.hi_new; g = k.e; }  // right member is node N+1
    const T t = q - p;
    if (e >= 0) uout[e] = fma(g, t, p);
    if (e + 1 < nx) uout[e + 1] = fma(-g, t, q);
}

template <typename T>
inline cudaError_t level_src_launch(const T* uin, T* uout, const T* src, int64_t nx, const Coef1<T>* coef,
                                    const SrcBc<T>& bc, int phase, cudaStream_t s) {
    const int64_t pairs = (nx + phase) / 2 + 1;   // left members -phase, 2-phase, ... <= nx-1
    const unsigned grid = (unsigned)((pairs + kSrcThreads - 1) / kSrcThreads);
    if (phase == 0) ge1d_level_src_kernel<T, 0><<<grid, kSrcThreads, 0, s>>>(uin, uout, src, nx, coef, bc);
    else            ge1d_level_src_kernel<T, 1><<<grid, kSrcThreads, 0, s>>>(uin, uout, src, nx, coef, bc);
    return cudaGetLastError();
}

}  // namespace ge
