// ge_level.cuh -- strategy A: one kernel launch per level, one HBM round trip
// per level.  Each thread owns V consecutive elements
// (one 16-byte vector, or V = 1 in the unaligned fallback), fetches the two
// previous-level neighbours on either side through L1 and writes its own
// outputs; a group that straddles two threads is evaluated by both, each
// keeping its own members (the kernel is HBM-bound, the ALUs are idle).
#pragma once
#include "ge_common.cuh"

namespace ge {

// ---------------------------------------------------------------- 1-D ------
// Value of element idx (0-based interior index; node idx+1) with the Dirichlet
// ghosts: element -1 is node 0, element nx is node N+1.
template <typename T>
__device__ __forceinline__ T fetch1(const T* __restrict__ in, int64_t idx, int64_t nx,
                                    const Coef1<T>& k) {
    if (idx < 0) return idx == -1 ? k.lo : T(0);
    if (idx >= nx) return idx == nx ? k.hi : T(0);
    return __ldg(in + idx);
}

constexpr int kLevelThreads = 256;

template <typename T, int V, int PH, int ITER>
__global__ void __launch_bounds__(kLevelThreads)
ge1d_level_kernel(const T* __restrict__ uin, T* __restrict__ uout, int64_t nx, int64_t batch,
                  const Coef1<T>* __restrict__ coef) {
    for (int64_t rod = blockIdx.y; rod < batch; rod += gridDim.y) {
        const Coef1<T> k = coef[rod];
        const T* __restrict__ in = uin + rod * nx;
        T* __restrict__ out = uout + rod * nx;
#pragma unroll
        for (int it = 0; it < ITER; ++it) {
            const int64_t e0 = (((int64_t)blockIdx.x * ITER + it) * kLevelThreads + threadIdx.x) * V;
            if (e0 >= nx) continue;
            // x[0..1] = e0-2, e0-1 ; x[2..V+1] = own ; x[V+2..V+3] = e0+V, e0+V+1
            T x[V + 4];
            if constexpr (V > 1) {
                T own[V], nb[V];
                ld_vec(in + e0, own);
#pragma unroll
                for (int j = 0; j < V; ++j) x[2 + j] = own[j];
                if (e0 >= V) { ld_vec(in + e0 - V, nb); x[0] = nb[V - 2]; x[1] = nb[V - 1]; }
                else { x[0] = T(0); x[1] = k.lo; }
                if (e0 + V < nx) { ld_vec(in + e0 + V, nb); x[V + 2] = nb[0]; x[V + 3] = nb[1]; }
                else { x[V + 2] = k.hi; x[V + 3] = T(0); }
            } else {
#pragma unroll
                for (int j = 0; j < V + 4; ++j) x[j] = fetch1(in, e0 - 2 + j, nx, k);
            }
            T o[V];
#pragma unroll
            for (int j = 0; j < V; ++j) {
                const int64_t e = e0 + j;
                // left members sit at elements e == PH (mod 2)
                const bool left = V > 1 ? (((j + PH) & 1) == 0) : (((e + PH) & 1) == 0);
                T lo, hi;
                if (left) {   // pair (e, e+1): needs e-1 .. e+2
                    pair_update_bc(x[j + 1], x[j + 2], x[j + 3], x[j + 4], k, false, e + 1 == nx, lo, hi);
                    o[j] = lo;
                } else {      // pair (e-1, e): needs e-2 .. e+1
                    pair_update_bc(x[j], x[j + 1], x[j + 2], x[j + 3], k, e == 0, false, lo, hi);
                    o[j] = hi;
                }
            }
            if constexpr (V > 1) st_vec(out + e0, o);
            else out[e0] = o[0];
        }
    }
}

// ---------------------------------------------------------------- 2-D ------
// DESIGN.md reading R-2D.  (x, y) are 0-based interior indices; the ghosts
// x = -1, x = nx, y = -1, y = ny carry the four edge values.
template <typename T>
__device__ __forceinline__ T ghost2(int64_t x, int64_t y, int64_t nx, int64_t ny, const Coef2<T>& k) {
    if (y < 0) return y == -1 ? k.ylo : T(0);
    if (y >= ny) return y == ny ? k.yhi : T(0);
    if (x < 0) return x == -1 ? k.xlo : T(0);
    return x == nx ? k.xhi : T(0);
}

// The 2x2 group.  w is the 4x4 previous-level window around the group
// (w[1][1]=a, w[1][2]=b, w[2][1]=c, w[2][2]=d; window corners unused).
// For an interior member P with out-of-group neighbours O1, O2:
//     R_P = u_P + r ((O1 - u_P) + (O2 - u_P))
// full group (eigenvectors (1,1,1,1):1, (1,0,0,-1),(0,1,-1,0):1+2r, (1,-1,-1,1):1+4r):
//     E1 = R_a - R_d, E2 = R_b - R_c, Q = (R_a + R_d) - (R_b + R_c)
//     a' = R_a - g2 E1 - g4 Q   d' = R_d + g2 E1 - g4 Q
//     b' = R_b - g2 E2 + g4 Q   c' = R_c + g2 E2 + g4 Q
// edge group, interior members m1, m2, in-group boundary value beta:
//     m1' = R_1 - h1 (R_1 + R_2 - 2 beta) - h3 (R_1 - R_2),  h1 = r/(2(1+r)), h3 = 3r/(2(1+3r))
// corner group, single member, boundary values bx, by:
//     m' = R - g2 (2R - bx - by)
// xg/yg: 0 = all members interior in that axis, 1 = low members are boundary nodes, 2 = high members.
template <typename T>
__device__ __forceinline__ void group_update(const T (&w)[4][4], const Coef2<T>& k, int xg, int yg,
                                             T& na, T& nb, T& nc, T& nd) {
    const T a = w[1][1], b = w[1][2], c = w[2][1], d = w[2][2];
    const T Ra = fma(k.r, (w[1][0] - a) + (w[0][1] - a), a);
    const T Rb = fma(k.r, (w[1][3] - b) + (w[0][2] - b), b);
    const T Rc = fma(k.r, (w[2][0] - c) + (w[3][1] - c), c);
    const T Rd = fma(k.r, (w[2][3] - d) + (w[3][2] - d), d);
    if (xg == 0 && yg == 0) {
        const T E1 = Ra - Rd, E2 = Rb - Rc;
        const T Q = (Ra + Rd) - (Rb + Rc);
        na = fma(-k.g4, Q, fma(-k.g2, E1, Ra));
        nd = fma(-k.g4, Q, fma(k.g2, E1, Rd));
        nb = fma(k.g4, Q, fma(-k.g2, E2, Rb));
        nc = fma(k.g4, Q, fma(k.g2, E2, Rc));
        return;
    }
    na = a; nb = b; nc = c; nd = d;
    if (xg != 0 && yg != 0) {           // corner: one interior member
        const T bx = xg == 1 ? k.xlo : k.xhi, by = yg == 1 ? k.ylo : k.yhi;
        const T R = xg == 1 ? (yg == 1 ? Rd : Rb) : (yg == 1 ? Rc : Ra);
        const T v = fma(-k.g2, (R - bx) + (R - by), R);
        if (xg == 1) { if (yg == 1) nd = v; else nb = v; }
        else         { if (yg == 1) nc = v; else na = v; }
        return;
    }
    T R1, R2, beta;
    if (xg != 0) {                      // members adjacent along y: (b,d) or (a,c)
        R1 = xg == 1 ? Rb : Ra; R2 = xg == 1 ? Rd : Rc; beta = xg == 1 ? k.xlo : k.xhi;
    } else {                            // members adjacent along x: (c,d) or (a,b)
        R1 = yg == 1 ? Rc : Ra; R2 = yg == 1 ? Rd : Rb; beta = yg == 1 ? k.ylo : k.yhi;
    }
    const T s = (R1 - beta) + (R2 - beta), df = R1 - R2;
    const T v1 = fma(-k.h3, df, fma(-k.h1, s, R1));
    const T v2 = fma(k.h3, df, fma(-k.h1, s, R2));
    if (xg == 1) { nb = v1; nd = v2; } else if (xg == 2) { na = v1; nc = v2; }
    else if (yg == 1) { nc = v1; nd = v2; } else { na = v1; nb = v2; }
}

constexpr int kLevel2dBx = 32, kLevel2dBy = 8;

// AL = false: rows of any length at any alignment -- the thread still owns V columns of a group row (so every group is
// computed once), read and written element by element; the last thread of a row may own fewer than V.
template <typename T, int V, int PH, bool AL = true>
__global__ void __launch_bounds__(kLevel2dBx * kLevel2dBy)
ge2d_level_kernel(const T* __restrict__ uin, T* __restrict__ uout, int64_t nx, int64_t ny,
                  const Coef2<T>* __restrict__ coef) {
    const Coef2<T> k = *coef;
    const int64_t e0 = ((int64_t)blockIdx.x * kLevel2dBx + threadIdx.x) * V;
    const int64_t j0 = 2 * ((int64_t)blockIdx.y * kLevel2dBy + threadIdx.y) - PH;   // anchor row
    if (e0 >= nx || j0 >= ny) return;

    // previous-level window: rows j0-1 .. j0+2, columns e0-2 .. e0+V+1
    T w[4][V + 4];
#pragma unroll
    for (int rr = 0; rr < 4; ++rr) {
        const int64_t y = j0 - 1 + rr;
        const bool yin = y >= 0 && y < ny;
        if constexpr (V > 1 && AL) {
            constexpr int NV = VecOf<T>::V;            // native 16-byte vector; V is a multiple of it
            T t[NV];
            if (yin) {
                const T* __restrict__ row = uin + y * nx;
#pragma unroll
                for (int c = 0; c < V / NV; ++c) {
                    ld_vec(row + e0 + c * NV, t);
#pragma unroll
                    for (int j = 0; j < NV; ++j) w[rr][2 + c * NV + j] = t[j];
                }
                if (e0 >= NV) { ld_vec(row + e0 - NV, t); w[rr][0] = t[NV - 2]; w[rr][1] = t[NV - 1]; }
                else { w[rr][0] = T(0); w[rr][1] = k.xlo; }
                if (e0 + V < nx) { ld_vec(row + e0 + V, t); w[rr][V + 2] = t[0]; w[rr][V + 3] = t[1]; }
                else { w[rr][V + 2] = k.xhi; w[rr][V + 3] = T(0); }
            } else {
#pragma unroll
                for (int j = 0; j < V + 4; ++j) w[rr][j] = ghost2(e0 - 2 + j, y, nx, ny, k);
            }
        } else {
#pragma unroll
            for (int j = 0; j < V + 4; ++j) {
                const int64_t x = e0 - 2 + j;
                w[rr][j] = (yin && x >= 0 && x < nx) ? __ldg(uin + y * nx + x) : ghost2(x, y, nx, ny, k);
            }
        }
    }

    const int yg = j0 < 0 ? 1 : (j0 + 1 >= ny ? 2 : 0);
    T o[2][V];
    // groups overlapping the columns e0 .. e0+V-1: anchors gx == PH (mod 2)
    const int first = V > 1 ? -PH : -(int)((e0 + PH) & 1);   // anchor offset of the first group
#pragma unroll
    for (int m = first; m < V; m += 2) {
        const int64_t gx = e0 + m;
        if (gx >= nx) continue;
        const int xg = gx < 0 ? 1 : (gx + 1 >= nx ? 2 : 0);
        T g[4][4];
#pragma unroll
        for (int rr = 0; rr < 4; ++rr)
#pragma unroll
            for (int cc = 0; cc < 4; ++cc) g[rr][cc] = w[rr][m + 1 + cc];   // columns gx-1 .. gx+2
        T na, nb, nc, nd;
        group_update(g, k, xg, yg, na, nb, nc, nd);
        if (m >= 0) { o[0][m] = na; o[1][m] = nc; }
        if (m + 1 < V) { o[0][m + 1] = nb; o[1][m + 1] = nd; }
    }
#pragma unroll
    for (int rr = 0; rr < 2; ++rr) {
        const int64_t y = j0 + rr;
        if (y < 0 || y >= ny) continue;
        if constexpr (V > 1 && AL) {
            constexpr int NV = VecOf<T>::V;
#pragma unroll
            for (int c = 0; c < V / NV; ++c) {
                T t[NV];
#pragma unroll
                for (int j = 0; j < NV; ++j) t[j] = o[rr][c * NV + j];
                st_vec(uout + y * nx + e0 + c * NV, t);
            }
        } else {
#pragma unroll
            for (int j = 0; j < V; ++j)
                if (e0 + j < nx) uout[y * nx + e0 + j] = o[rr][j];
        }
    }
}

}  // namespace ge
