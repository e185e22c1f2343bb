// ge_level_var.cuh -- strategy A (1-D, two-point groups) with VARIABLE DIFFUSIVITY (
// DESIGN.md reading R-VAR):  u_t = (a(x) u_x)_x  in flux form, one number per link,
//     rl[j] = tau a_{j+1/2} / h^2   for the link between nodes j and j+1,  j = 0 .. N.
// The paper's model problem has a constant coefficient; PAPER.md:37 names diffusion steps inside an
// operator splitting of transport equations as the use.
//
// A pair (i, i+1) takes the flux through its inner link rm = rl[i] at the new level and through its outer links
// rl[i-1], rl[i+1] at the old level; the 2x2 block [[1+rm, -rm], [-rm, 1+rm]] keeps the eigenvalues 1 and 1+2rm, so
// the factored form of ge_common.cuh carries over with per-link coefficients:
//     p = u_i + rl[i-1] (u_{i-1} - u_i),  q = u_{i+1} + rl[i+1] (u_{i+2} - u_{i+1}),  w = rm/(1+2rm) (q - p),
//     new_i = p + w,  new_{i+1} = q - w.
// A pair with a boundary member: that unknown is pinned to the Dirichlet value, rm/(1+2rm) becomes rm/(1+rm).
// One thread per pair; HBM sees u in, rl in, u out: 3 * sizeof(T) algorithmic bytes per update.
#pragma once
#include "ge_common.cuh"

namespace ge {

constexpr int kVarThreads = 256;

template <typename T, int PH>
__global__ void __launch_bounds__(kVarThreads)
ge1d_level_var_kernel(const T* __restrict__ uin, T* __restrict__ uout, const T* __restrict__ rl, int64_t nx,
                      const Coef1<T>* __restrict__ coef) {
    const int64_t m = (int64_t)blockIdx.x * kVarThreads + threadIdx.x;
    const int64_t e = 2 * m - PH;                 // element of the pair's left member (-1: node 0); node = element + 1
    if (e >= nx) return;
    const T lo = coef->lo, hi = coef->hi;
    auto old = [&](int64_t i) -> T {              // element i of the old level, boundaries at -1 and nx
        if (i < 0) return lo;
        if (i >= nx) return hi;
        return __ldg(uin + i);
    };
    const T a = old(e - 1), b = old(e), c = old(e + 1), d = old(e + 2);
    const T rm = __ldg(rl + e + 1);                                   // inner link: nodes e+1, e+2
    T p = e >= 0 ? fma(__ldg(rl + e), a - b, b) : lo;                 // outer link to the left: nodes e, e+1
    T q = e + 1 < nx ? fma(__ldg(rl + e + 2), d - c, c) : hi;         // outer link to the right: nodes e+2, e+3
    const bool cut = e < 0 || e + 1 >= nx;
    const T g = rm / (cut ? T(1) + rm : fma(T(2), rm, T(1)));
    const T t = q - p;
    if (e >= 0) uout[e] = fma(g, t, p);
    if (e + 1 < nx) uout[e + 1] = fma(-g, t, q);
}

template <typename T>
inline cudaError_t level_var_launch(const T* uin, T* uout, const T* rl, int64_t nx, const Coef1<T>* coef, int phase,
                                    cudaStream_t s) {
    const int64_t pairs = (nx + phase) / 2 + 1;   // left members -phase, 2-phase, ... <= nx-1
    const unsigned grid = (unsigned)((pairs + kVarThreads - 1) / kVarThreads);
    if (phase == 0) ge1d_level_var_kernel<T, 0><<<grid, kVarThreads, 0, s>>>(uin, uout, rl, nx, coef);
    else            ge1d_level_var_kernel<T, 1><<<grid, kVarThreads, 0, s>>>(uin, uout, rl, nx, coef);
    return cudaGetLastError();
}

}  // namespace ge
