// ge_common.cuh -- shared device helpers of libge (sm_100a).
//
// Arithmetic form.  The kernels never use the four printed weights of
// PAPER.md Eqs (3),(4): they use the algebraically equal FACTORED form
//
//     p = u_i     + r (u_{i-1} - u_i)          Saul'yev right-hand side of Eq (2) at i
//     q = u_{i+1} + r (u_{i+2} - u_{i+1})      Saul'yev right-hand side of Eq (1) at i+1
//     w = g (q - p),  g = r/(1+2r);   new_i = p + w,  new_{i+1} = q - w
// (the 2x2 block [[1+r,-r],[-r,1+r]] has eigenvalues 1 and 1+2r: the mean of
// (p,q) passes, the difference is divided by 1+2r).  A pair with a boundary
// member is the same system with one unknown pinned to beta:
//     partner of node 1 is node 0:    new_1 = q - e (q - beta_lo),  e = r/(1+r)   (Eq (1))
//     partner of node N is node N+1:  new_N = p + e (beta_hi - p)                 (Eq (2))
// Each update is "value + small correction", which keeps fp32 within 1e-5 of
// the fp64 oracle over thousands of levels where rounded weights drift.
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

namespace ge {

// Per-rod coefficients, computed in fp64 on the host, rounded once to T.
template <typename T>
struct Coef1 {
    T r;     // tau/h^2
    T g;     // r/(1+2r)
    T e;     // r/(1+r)
    T lo;    // u at node 0
    T hi;    // u at node N+1
    T pad[3];
};

// 2-D coefficients (one set per plan).
template <typename T>
struct Coef2 {
    T r;
    T g2;    // r/(1+2r)
    T g4;    // r/(1+4r)
    T h1;    // r/(2(1+r))     edge groups: mean mode
    T h3;    // 3r/(2(1+3r))   edge groups: difference mode
    T xlo, xhi, ylo, yhi;   // edge values
    T pad[7];
};

// 3-D coefficients (one set per plan; ge_level3d.cuh).
template <typename T>
struct Coef3 {
    T r;
    T c1, c2, c3;          // 2r/(1+2r)/8, 4r/(1+4r)/8, 6r/(1+6r)/8
    T lo[3], hi[3];        // face values: x, y, z
    T q1, q2, q3;          // group cut by ONE face (4 members): r/(1+r)/4, 3r/(1+3r)/4, 5r/(1+5r)/4
    T pad[3];
};

template <typename T> struct VecOf;
template <> struct VecOf<float>  { using type = float4;  static constexpr int V = 4; };
template <> struct VecOf<double> { using type = double2; static constexpr int V = 2; };

template <typename T>
__device__ __forceinline__ void ld_vec(const T* __restrict__ p, T (&x)[VecOf<T>::V]) {
    using VT = typename VecOf<T>::type;
    VT v = __ldg(reinterpret_cast<const VT*>(p));
    if constexpr (VecOf<T>::V == 4) { x[0] = v.x; x[1] = v.y; x[2] = v.z; x[3] = v.w; }
    else { x[0] = v.x; x[1] = v.y; }
}

template <typename T>
__device__ __forceinline__ void st_vec(T* __restrict__ p, const T (&x)[VecOf<T>::V]) {
    using VT = typename VecOf<T>::type;
    VT v;
    if constexpr (VecOf<T>::V == 4) { v.x = x[0]; v.y = x[1]; v.z = x[2]; v.w = x[3]; }
    else { v.x = x[0]; v.y = x[1]; }
    *reinterpret_cast<VT*>(p) = v;
}

// The two-point group: from level-n values (a,b,c,d) = u_{i-1}, u_i, u_{i+1}, u_{i+2}
// produce level-(n+1) u_i (lo) and u_{i+1} (hi).   PAPER.md:94-104 (Eqs 3,4), factored.
template <typename T>
__device__ __forceinline__ void pair_update(T a, T b, T c, T d, T r, T g, T& lo, T& hi) {
    const T p = fma(r, a - b, b);
    const T q = fma(r, d - c, c);
    const T t = q - p;
    lo = fma(g, t, p);
    hi = fma(-g, t, q);
}

// Same with the boundary-truncated cases folded in:
//   b_is_bc: member i is node 0     -> p := beta_lo, g := e   (only `hi` is meaningful)
//   c_is_bc: member i+1 is node N+1 -> q := beta_hi, g := e   (only `lo` is meaningful)
template <typename T>
__device__ __forceinline__ void pair_update_bc(T a, T b, T c, T d, const Coef1<T>& k,
                                               bool b_is_bc, bool c_is_bc, T& lo, T& hi) {
    T p = fma(k.r, a - b, b);
    T q = fma(k.r, d - c, c);
    T g = k.g;
    if (b_is_bc) { p = k.lo; g = k.e; }
    if (c_is_bc) { q = k.hi; g = k.e; }
    const T t = q - p;
    lo = fma(g, t, p);
    hi = fma(-g, t, q);
}

// Slide a lane's register window right by one element: slot j takes slot j+1, the last slot takes
// the next lane's slot 0 (lane 31 keeps a stale value there; the tile geometry accounts for it).
template <typename T, int C>
__device__ __forceinline__ void shift_window(T (&v)[C]) {
    const T t = __shfl_down_sync(0xffffffffu, v[0], 1);
#pragma unroll
    for (int j = 0; j + 1 < C; ++j) v[j] = v[j + 1];
    v[C - 1] = t;
}

}  // namespace ge
