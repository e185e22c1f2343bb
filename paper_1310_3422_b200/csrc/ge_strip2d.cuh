// ge_strip2d.cuh -- strategy B (2-D), drift-free: TB levels per HBM round trip,
// state in registers, no shared memory, no barrier.
//
// Scheme: DESIGN.md reading R-2D (2x2 four-point groups, anchors shifted by
// (1,1) between levels; PAPER.md:134, :228 only claim the extension).
//
// Like ge_temporal2d.cuh a WARP owns a strip of 32*C columns and streams along
// y through a pipeline of TB stages (stage l turns level-l row pairs into
// level-(l+1) row pairs, shifted down by one row -- the (0,1) part of the
// pattern's diagonal shift).  What is new is the x direction and the plumbing:
//   * x alternates R / L like the 1-D drift-free level pair (ge_resident.cuh):
//     a launch always starts at a phase-1 level, even stages are R (groups at
//     window slots (1,2) ... (C-1,C); the last group's right members come from
//     the next lane: two shuffles; results form the window shifted right by
//     one column), odd stages are L (groups at (-1,0) ... (C-3,C-2) of the
//     shifted window; the first group's left members come from the previous
//     lane; results are back in the unshifted window).  No realignment
//     shifts, no window drift, TB even.
//   * strips are aligned like the 1-D tiles: strip 0 starts at column 0, the
//     last strip ends at column nx-1, strips in between carry TB stale columns
//     per side.  A Dirichlet column never sits inside a lane; the x-edge groups
//     are a few selects on lane 0 / lane 31 of the first / last strip (BC),
//     compiled out for interior strips.  In the shifted state column 0 of the
//     first strip lives in one extra register per row.
//   * the row loop is unrolled by two, so the rotating row registers
//     (prev[l] <- cur) rotate by renaming, and row pairs are prefetched two
//     iterations ahead.
//   * groups cut by a y edge (and rows outside the grid) take a generic
//     out-of-line path built on ge_level.cuh group_update.
// Arithmetic: 6.75 flop-instructions per node update, the expression tree of
// ge2d_level_kernel (bit-identical results).
#pragma once
#include "ge_common.cuh"
#include "ge_level.cuh"

namespace ge {

constexpr int kStripWarps = 4;        // warps per CTA = adjacent strips (their halos share L2 lines)

struct Strip2dGeom {
    int halo;        // stale columns per side of an interior strip (multiple of V)
    int valid;       // output columns per strip
    int nreg;        // left-aligned + regular strips; strip nreg is the right-aligned last one
    int nstrips;     // nreg + 1
    int hp;          // output row pairs per segment
    int segs;
};

inline Strip2dGeom strip2d_geom(int C, int V, int TB, int64_t nx, int64_t ny, int hp) {
    Strip2dGeom g;
    g.halo = (TB + V - 1) / V * V;
    g.valid = 32 * C - 2 * g.halo;
    g.nreg = 1 + (int)((nx + g.halo - 32 * (int64_t)C) / g.valid);
    g.nstrips = g.nreg + 1;
    g.hp = hp;
    g.segs = (int)((ny + 2 * (int64_t)hp - 1) / (2 * (int64_t)hp));
    return g;
}

template <typename T>
struct Strip2dCtx {
    T r, g2, g4, h1, h3, xlo, xhi;
    bool is_lo, is_hi;     // this lane holds column 0 in slot 0 / column nx-1 in slot C-1 (unshifted)
};

// the closed-form 4x4 solve, members a b / c d
template <typename T>
__device__ __forceinline__ void solve4(T ra, T rb, T rc, T rd, T g2, T g4, T& na, T& nb, T& nc, T& nd) {
    const T E1 = ra - rd, E2 = rb - rc;
    const T Q = (ra + rd) - (rb + rc);
    na = fma(-g4, Q, fma(-g2, E1, ra));
    nd = fma(-g4, Q, fma(g2, E1, rd));
    nb = fma(g4, Q, fma(-g2, E2, rb));
    nc = fma(g4, Q, fma(g2, E2, rc));
}
// x-edge group: two interior members r1 (lower row), r2 (upper row), in-group boundary value beta
template <typename T>
__device__ __forceinline__ void solve2(T r1, T r2, T beta, T h1, T h3, T& n1, T& n2) {
    const T s = (r1 - beta) + (r2 - beta), df = r1 - r2;
    n1 = fma(-h3, df, fma(-h1, s, r1));
    n2 = fma(h3, df, fma(-h1, s, r2));
}

// right-hand sides of the columns in slots 2m (right members b, d of the group to the left) and
// 2m+1 (left members a, c) for the group rows (P1, Q0); P0 / Q1 are the rows below / above
template <typename T, int C>
__device__ __forceinline__ void strip_rhs(const T (&P0)[C], const T (&P1)[C], const T (&Q0)[C], const T (&Q1)[C],
                                          T r, T (&Ra)[C / 2], T (&Rb)[C / 2], T (&Rc)[C / 2], T (&Rd)[C / 2]) {
#pragma unroll
    for (int m = 0; m < C / 2; ++m) {
        const T exP = P1[2 * m + 1] - P1[2 * m];
        const T exQ = Q0[2 * m + 1] - Q0[2 * m];
        const T eyLb = P1[2 * m] - P0[2 * m], eyLa = P1[2 * m + 1] - P0[2 * m + 1];
        const T eyHd = Q1[2 * m] - Q0[2 * m], eyHc = Q1[2 * m + 1] - Q0[2 * m + 1];
        Rb[m] = fma(r, exP - eyLb, P1[2 * m]);          // right + below
        Rd[m] = fma(r, exQ + eyHd, Q0[2 * m]);          // right + above
        Ra[m] = fma(-r, exP + eyLa, P1[2 * m + 1]);     // left + below
        Rc[m] = fma(r, eyHc - exQ, Q0[2 * m + 1]);      // left + above
    }
}

// R: unshifted rows -> rows shifted right by one column.  N0 / N1 are the new rows of P1 / Q0;
// nx0[0..1]: new column 0 of those rows (lane is_lo only).
template <typename T, int C, bool BC>
__device__ __forceinline__ void strip_stage_R(const T (&P0)[C], const T (&P1)[C], const T (&Q0)[C],
                                              const T (&Q1)[C], T (&N0)[C], T (&N1)[C], T (&nx0)[2],
                                              const Strip2dCtx<T>& k) {
    constexpr unsigned FULL = 0xffffffffu;
    T Ra[C / 2], Rb[C / 2], Rc[C / 2], Rd[C / 2];
    strip_rhs<T, C>(P0, P1, Q0, Q1, k.r, Ra, Rb, Rc, Rd);
    const T RbN = __shfl_down_sync(FULL, Rb[0], 1);
    const T RdN = __shfl_down_sync(FULL, Rd[0], 1);
#pragma unroll
    for (int m = 0; m < C / 2; ++m) {
        const T rb = m + 1 < C / 2 ? Rb[m + 1] : RbN;
        const T rd = m + 1 < C / 2 ? Rd[m + 1] : RdN;
        T na, nb, nc, nd;
        solve4(Ra[m], rb, Rc[m], rd, k.g2, k.g4, na, nb, nc, nd);
        if constexpr (BC) {
            if (m == C / 2 - 1 && k.is_hi) {       // members b, d are the boundary column x = nx
                solve2(Ra[m], Rc[m], k.xhi, k.h1, k.h3, na, nc);
                nb = k.xhi; nd = k.xhi;
            }
        }
        N0[2 * m] = na; N0[2 * m + 1] = nb;
        N1[2 * m] = nc; N1[2 * m + 1] = nd;
    }
    if constexpr (BC) solve2(Rb[0], Rd[0], k.xlo, k.h1, k.h3, nx0[0], nx0[1]);   // group (x = -1, 0)
}

// L: rows shifted right by one column -> unshifted rows.  pP / pQ: column 0 of the rows
// P0, P1 / Q0, Q1 (lane is_lo only).
template <typename T, int C, bool BC>
__device__ __forceinline__ void strip_stage_L(const T (&P0)[C], const T (&P1)[C], const T (&Q0)[C],
                                              const T (&Q1)[C], const T (&pP)[2], const T (&pQ)[2],
                                              T (&N0)[C], T (&N1)[C], const Strip2dCtx<T>& k) {
    constexpr unsigned FULL = 0xffffffffu;
    T Ra[C / 2], Rb[C / 2], Rc[C / 2], Rd[C / 2];
    strip_rhs<T, C>(P0, P1, Q0, Q1, k.r, Ra, Rb, Rc, Rd);
    T ra = __shfl_up_sync(FULL, Ra[C / 2 - 1], 1);
    T rc = __shfl_up_sync(FULL, Rc[C / 2 - 1], 1);
    if constexpr (BC) {
        if (k.is_lo) {     // members a, c are column 0; their left neighbour is the boundary column
            const T a = pP[1], c = pQ[0];
            ra = fma(-k.r, (a - k.xlo) + (a - pP[0]), a);
            rc = fma(k.r, (pQ[1] - c) - (c - k.xlo), c);
        }
    }
    solve4(ra, Rb[0], rc, Rd[0], k.g2, k.g4, N0[0], N0[1], N1[0], N1[1]);
#pragma unroll
    for (int m = 0; m + 1 < C / 2; ++m)
        solve4(Ra[m], Rb[m + 1], Rc[m], Rd[m + 1], k.g2, k.g4, N0[2 * m + 2], N0[2 * m + 3], N1[2 * m + 2],
               N1[2 * m + 3]);
}

// Generic stage for the few stage-iterations whose group rows (j, j+1) are not both interior
// rows.  ext: rows P0, P1, Q0, Q1 with window slots -2 .. C+1 (ext[row][slot + 2]); o: new rows of
// P1 / Q0 in the OUTPUT window (R: slot s = input slot s+1; L: slot s = input slot s-1), then
// o[2*C], o[2*C+1] = new column 0 of the two rows (R, lane is_lo).
// yg: 1 the lower group row is the boundary row y = -1, 2 the upper one is y = ny, 0 neither;
// outside: both rows lie outside the grid (values are carried, boundary rows stay pinned).
template <typename T, int C, bool SHIFTED>
__device__ __noinline__ void strip_stage_edge(const T* __restrict__ ext, T* __restrict__ o,
                                              const Coef2<T>* __restrict__ kp, int yg, bool outside,
                                              bool is_lo, bool is_hi) {
    const Coef2<T> k = *kp;
    constexpr int E = C + 4;
    // groups of this lane: R (unshifted input) slots (2m+1, 2m+2), L (shifted input) slots (2m-1, 2m)
#pragma unroll
    for (int m = 0; m < C / 2; ++m) {
        const int s0 = SHIFTED ? 2 * m - 1 : 2 * m + 1;          // slot of members a, c
        T w[4][4];
#pragma unroll
        for (int rr = 0; rr < 4; ++rr)
#pragma unroll
            for (int cc = 0; cc < 4; ++cc) w[rr][cc] = ext[rr * E + (s0 - 1 + cc) + 2];
        T na = w[1][1], nb = w[1][2], nc = w[2][1], nd = w[2][2];
        if (!outside) {
            const int xg = (!SHIFTED && is_hi && m == C / 2 - 1) ? 2 : 0;
            group_update(w, k, xg, yg, na, nb, nc, nd);
        }
        if (!SHIFTED && is_hi && m == C / 2 - 1) { nb = k.xhi; nd = k.xhi; }   // the boundary column stays pinned
        const int so = SHIFTED ? 2 * m : 2 * m;                  // output slots of a, b
        o[so] = na; o[so + 1] = nb;
        o[C + so] = nc; o[C + so + 1] = nd;
    }
    if (!SHIFTED) {
        // lane is_lo: the group (x = -1, 0), members a, c on the boundary column
        T w[4][4];
#pragma unroll
        for (int rr = 0; rr < 4; ++rr)
#pragma unroll
            for (int cc = 0; cc < 4; ++cc) w[rr][cc] = ext[rr * E + (-2 + cc) + 2];
        T na = w[1][1], nb = w[1][2], nc = w[2][1], nd = w[2][2];
        if (!outside && is_lo) group_update(w, k, 1, yg, na, nb, nc, nd);
        o[2 * C] = nb; o[2 * C + 1] = nd;
    }
}

// Builds the extended rows (two neighbour columns per side) and runs the generic stage.
template <typename T, int C, bool SHIFTED, bool BC>
__device__ __forceinline__ void strip_stage_slow(const T (&P0)[C], const T (&P1)[C], const T (&Q0)[C],
                                                 const T (&Q1)[C], const T (&pP)[2], const T (&pQ)[2],
                                                 T (&N0)[C], T (&N1)[C], T (&nx0)[2], const Strip2dCtx<T>& k,
                                                 const Coef2<T>* __restrict__ coef, int yg, bool outside) {
    constexpr unsigned FULL = 0xffffffffu;
    constexpr int E = C + 4;
    T ext[4 * E];
    const T* rows[4] = {P0, P1, Q0, Q1};
    const T col0[4] = {pP[0], pP[1], pQ[0], pQ[1]};
#pragma unroll
    for (int rr = 0; rr < 4; ++rr) {
        const T* v = rows[rr];
#pragma unroll
        for (int s = 0; s < C; ++s) ext[rr * E + s + 2] = v[s];
        T l2 = __shfl_up_sync(FULL, v[C - 2], 1), l1 = __shfl_up_sync(FULL, v[C - 1], 1);
        T r0 = __shfl_down_sync(FULL, v[0], 1), r1 = __shfl_down_sync(FULL, v[1], 1);
        if (BC && k.is_lo) {
            if (SHIFTED) { l1 = col0[rr]; l2 = k.xlo; } else { l1 = k.xlo; l2 = T(0); }
        }
        if (BC && k.is_hi) {
            if (SHIFTED) { r0 = T(0); r1 = T(0); } else { r0 = k.xhi; r1 = T(0); }
        }
        ext[rr * E + 0] = l2; ext[rr * E + 1] = l1;
        ext[rr * E + C + 2] = r0; ext[rr * E + C + 3] = r1;
    }
    T o[2 * C + 2];
    strip_stage_edge<T, C, SHIFTED>(ext, o, coef, yg, outside, BC && k.is_lo, BC && k.is_hi);
#pragma unroll
    for (int s = 0; s < C; ++s) { N0[s] = o[s]; N1[s] = o[C + s]; }
    if (!SHIFTED) { nx0[0] = o[2 * C]; nx0[1] = o[2 * C + 1]; }
}

// Row y of the lane's columns [e0, e0+C); rows outside the grid return the boundary value (y = -1,
// y = ny) or a finite filler.  The strip lies inside the grid in x, so every load is a full vector.
template <typename T, int C>
__device__ __forceinline__ void strip_load_row(const T* __restrict__ uin, int nx, int ny, T ylo, T yhi, int y,
                                               int e0, T (&v)[C]) {
    constexpr int V = VecOf<T>::V;
    if ((unsigned)y < (unsigned)ny) {
        const T* __restrict__ row = uin + (int64_t)y * nx + e0;
#pragma unroll
        for (int c = 0; c < C / V; ++c) {
            T t[V];
            ld_vec(row + c * V, t);
#pragma unroll
            for (int j = 0; j < V; ++j) v[c * V + j] = t[j];
        }
    } else {
        const T f = y == -1 ? ylo : (y == ny ? yhi : T(0));
#pragma unroll
        for (int j = 0; j < C; ++j) v[j] = f;
    }
}

template <typename T, int C, int TB, bool BC>
__device__ __forceinline__ void strip_run(const T* __restrict__ uin, T* __restrict__ uout, int nx, int ny,
                                          const Coef2<T>* __restrict__ coef, int a0, int out_lo, int out_hi,
                                          bool first, bool last, int ys, int ye, int lane) {
    constexpr int V = VecOf<T>::V;
    static_assert(TB % 2 == 0 && C % 2 == 0 && C % V == 0, "TB even; C holds whole groups and vectors");
    const Coef2<T> kk = *coef;
    Strip2dCtx<T> k;
    k.r = kk.r; k.g2 = kk.g2; k.g4 = kk.g4; k.h1 = kk.h1; k.h3 = kk.h3; k.xlo = kk.xlo; k.xhi = kk.xhi;
    k.is_lo = BC && first && lane == 0; k.is_hi = BC && last && lane == 31;
    const int e0 = a0 + lane * C;
    const int Y0 = ys - TB;                       // first row pair that enters the pipeline
    const int iters = (ye - ys + 1) / 2 + TB;

    T prev[TB][2][C];
    T px[TB][2];                                  // column 0 of prev[l] (odd l: shifted rows; lane is_lo)
#pragma unroll
    for (int l = 0; l < TB; ++l) {
#pragma unroll
        for (int j = 0; j < C; ++j) { prev[l][0][j] = T(0); prev[l][1][j] = T(0); }
        px[l][0] = T(0); px[l][1] = T(0);
    }
    T L0[2][C], L1[2][C];                         // row pairs in flight, two iterations ahead
    strip_load_row<T, C>(uin, nx, ny, kk.ylo, kk.yhi, Y0, e0, L0[0]);
    strip_load_row<T, C>(uin, nx, ny, kk.ylo, kk.yhi, Y0 + 1, e0, L0[1]);
    strip_load_row<T, C>(uin, nx, ny, kk.ylo, kk.yhi, Y0 + 2, e0, L1[0]);
    strip_load_row<T, C>(uin, nx, ny, kk.ylo, kk.yhi, Y0 + 3, e0, L1[1]);

    auto body = [&](int it, T (&LL)[2][C]) {
        const int y0 = Y0 + 2 * it;
        T cur[2][C], cx[2] = {T(0), T(0)};
#pragma unroll
        for (int s = 0; s < C; ++s) { cur[0][s] = LL[0][s]; cur[1][s] = LL[1][s]; }
        strip_load_row<T, C>(uin, nx, ny, kk.ylo, kk.yhi, y0 + 4, e0, LL[0]);
        strip_load_row<T, C>(uin, nx, ny, kk.ylo, kk.yhi, y0 + 5, e0, LL[1]);
#pragma unroll
        for (int l = 0; l < TB; ++l) {
            const int j = y0 - 1 - l;             // lower row of this stage's groups
            T nw[2][C], nwx[2] = {T(0), T(0)};
            if ((unsigned)j < (unsigned)(ny - 1)) {
                if (l % 2 == 0) strip_stage_R<T, C, BC>(prev[l][0], prev[l][1], cur[0], cur[1], nw[0], nw[1], nwx, k);
                else            strip_stage_L<T, C, BC>(prev[l][0], prev[l][1], cur[0], cur[1], px[l], cx, nw[0], nw[1], k);
            } else {
                const int yg = j == -1 ? 1 : (j + 1 == ny ? 2 : 0);
                if (l % 2 == 0)
                    strip_stage_slow<T, C, false, BC>(prev[l][0], prev[l][1], cur[0], cur[1], px[l], cx, nw[0],
                                                      nw[1], nwx, k, coef, yg, yg == 0);
                else
                    strip_stage_slow<T, C, true, BC>(prev[l][0], prev[l][1], cur[0], cur[1], px[l], cx, nw[0],
                                                     nw[1], nwx, k, coef, yg, yg == 0);
            }
#pragma unroll
            for (int s = 0; s < C; ++s) {
                prev[l][0][s] = cur[0][s]; prev[l][1][s] = cur[1][s];
                cur[0][s] = nw[0][s]; cur[1][s] = nw[1][s];
            }
            if constexpr (BC) { px[l][0] = cx[0]; px[l][1] = cx[1]; cx[0] = nwx[0]; cx[1] = nwx[1]; }
        }
        // cur holds level-TB rows (y0 - TB, y0 - TB + 1), unshifted (TB is even)
        if (it >= TB) {
            const int yo = y0 - TB;
#pragma unroll
            for (int rr = 0; rr < 2; ++rr) {
                if (yo + rr < ye) {
                    T* __restrict__ row = uout + (int64_t)(yo + rr) * nx;
#pragma unroll
                    for (int c = 0; c < C / V; ++c) {
                        const int e = e0 + c * V;
                        if (e >= out_lo && e < out_hi) {
                            T t[V];
#pragma unroll
                            for (int q = 0; q < V; ++q) t[q] = cur[rr][c * V + q];
                            st_vec(row + e, t);
                        }
                    }
                }
            }
        }
    };
#pragma unroll 1
    for (int it = 0; it < iters; it += 2) {
        body(it, L0);
        if (it + 1 < iters) body(it + 1, L1);
    }
}

template <typename T, int C, int TB>
__global__ void __launch_bounds__(kStripWarps * 32)
ge2d_strip_kernel(const T* __restrict__ uin, T* __restrict__ uout, int nx, int ny,
                  const Coef2<T>* __restrict__ coef, const Strip2dGeom g) {
    const int lane = threadIdx.x & 31;
    const int warp = threadIdx.x >> 5;
    const int strip = blockIdx.x * kStripWarps + warp;
    if (strip >= g.nstrips) return;
    const bool first = strip == 0, last = strip == g.nreg;
    const int a0 = first ? 0 : (last ? nx - 32 * C : strip * g.valid - g.halo);
    const int out_lo = strip * g.valid;
    const int out_hi = last ? nx : out_lo + g.valid;
    const int ys = 2 * g.hp * (int)blockIdx.y;
    const int ye = ys + 2 * g.hp < ny ? ys + 2 * g.hp : ny;
    if (first || last) strip_run<T, C, TB, true>(uin, uout, nx, ny, coef, a0, out_lo, out_hi, first, last, ys, ye, lane);
    else               strip_run<T, C, TB, false>(uin, uout, nx, ny, coef, a0, out_lo, out_hi, false, false, ys, ye, lane);
}

// Host launcher: TB levels starting at a PHASE-1 level.  Requires nx % V == 0, nx even, nx >= 32*C,
// 16-byte aligned buffers and nx, ny < 2^30.
template <typename T, int C, int TB>
inline cudaError_t strip2d_launch(const T* uin, T* uout, int64_t nx, int64_t ny, const Coef2<T>* coef, int hp,
                                  cudaStream_t s) {
    const Strip2dGeom g = strip2d_geom(C, VecOf<T>::V, TB, nx, ny, hp);
    dim3 grid((unsigned)((g.nstrips + kStripWarps - 1) / kStripWarps), (unsigned)g.segs);
    ge2d_strip_kernel<T, C, TB><<<grid, kStripWarps * 32, 0, s>>>(uin, uout, (int)nx, (int)ny, coef, g);
    return cudaGetLastError();
}

}  // namespace ge
