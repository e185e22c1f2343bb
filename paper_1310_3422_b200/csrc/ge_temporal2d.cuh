// ge_temporal2d.cuh -- strategy B (2-D): TB levels per launch, one HBM round
// trip per TB levels, state held in registers, no shared memory and no barrier.
//
// Scheme: DESIGN.md reading R-2D (2x2 four-point groups, anchors shifted by
// (1,1) between levels; PAPER.md:134, :228 only claim the extension).
//
// Decomposition.  A WARP owns a strip of 32*C columns and streams along y over
// one segment of rows ("2.5-D" temporal blocking).  Lane t holds C consecutive
// columns of every row in flight.  The rows travel through a pipeline of TB
// stages, stage l turning level-l rows into level-(l+1) rows:
//   * rows move in PAIRS.  Stage l receives the pair (y, y+1), still holds the
//     previous pair (y-2, y-1), and updates the groups whose rows are
//     (y-1, y): their 4x4 neighbourhood minus corners is exactly those four
//     rows.  Its output pair (y-1, y) is shifted down by one row against its
//     input -- which is precisely the (0,1) part of the pattern's diagonal
//     shift, so the next stage finds ITS groups aligned the same way.  Every
//     stage is the same code; after TB stages the pair has moved TB rows.
//   * in x the window slides exactly as in the 1-D kernel (ge_temporal.cuh):
//     the lane's groups have their left columns at window slots 1, 3, ...;
//     the results form the window shifted right by one column, which is where
//     the next level's groups sit.  `pre`/`post` realign to 16 bytes.
// A strip that started with 32*C columns keeps 32*C - 2*TB valid ones; a
// segment reads TB extra row pairs.  Per lane and stage one exchange: the lane
// computes the right-hand sides R of its slot-0 column (members of the LEFT
// neighbour's last group) and hands them over with two shuffles.
//
// Arithmetic (6.75 flops per node update; bit-identical to ge2d_level_kernel):
//   ex = difference across the vertical group boundary  (shared by 2 groups)
//   ey = difference across the horizontal group boundary
//   R_P = u_P + r (sum of the two out-of-group differences)
//   E1 = R_a - R_d, E2 = R_b - R_c, Q = (R_a + R_d) - (R_b + R_c)
//   a' = R_a - g2 E1 - g4 Q, d' = R_d + g2 E1 - g4 Q, b' = R_b - g2 E2 + g4 Q, c' = R_c + g2 E2 + g4 Q
// Groups cut by a Dirichlet edge: x-edges are patched per lane (only the lane
// that holds the ghost column diverges); y-edges take a generic out-of-line
// path (ge_level.cuh group_update) on the few stage-iterations that touch
// them.  Ghost rows/columns are carried as data and re-pinned every level.
#pragma once
#include "ge_common.cuh"
#include "ge_level.cuh"

namespace ge {

constexpr int kTemporal2dWarps = 4;   // warps per CTA = adjacent strips (their halos share L1/L2 lines)

struct Temporal2dGeom {
    int pre, post, shift;   // x realignment as in 1-D; shift = pre + TB + post
    int valid;              // output columns per strip (multiple of V)
    int hp;                 // output row pairs per segment
    int ybase;              // first output row of segment 0 (-1 or 0: parity of the last level's groups)
    int strips, segs;
};

inline Temporal2dGeom temporal2d_geom(int C, int V, int TB, int phase, int64_t nx, int64_t ny, int hp) {
    Temporal2dGeom g;
    g.pre = phase == 0 ? 1 : 0;
    g.post = (V - (g.pre + TB) % V) % V;
    g.shift = g.pre + TB + g.post;
    const int v = 32 * C - 2 * TB - 2 * g.pre - g.post;   // see temporal1d_geom
    g.valid = v - v % V;
    g.hp = hp;
    // stage 0's group rows are (Y0+1+2k, Y0+2+2k) with anchor parity == phase; Y0 = ybase - TB
    g.ybase = ((phase + 1 + TB) & 1) ? -1 : 0;
    g.strips = (int)((nx + g.valid - 1) / g.valid);
    g.segs = (int)((ny - g.ybase + 2 * (int64_t)hp - 1) / (2 * (int64_t)hp));
    return g;
}

// Generic stage for the stage-iterations whose group rows (j, j+1) are not both interior rows.
// win: rows j-1 .. j+2, window slots 0 .. C+1 (slots C, C+1 come from the next lane).
// o[0] = new row j, o[1] = new row j+1 in the shifted window (new slot s = old slot s+1).
template <typename T, int C, bool EX>
__device__ __noinline__ void temporal2d_stage_edge(const T* __restrict__ win, T* __restrict__ o,
                                                   const Coef2<T>* __restrict__ kp, int glo, int ghi, int yg,
                                                   bool outside) {
    const Coef2<T> k = *kp;
#pragma unroll
    for (int m = 0; m < C / 2; ++m) {
        T w[4][4];
#pragma unroll
        for (int rr = 0; rr < 4; ++rr)
#pragma unroll
            for (int cc = 0; cc < 4; ++cc) w[rr][cc] = win[rr * (C + 2) + 2 * m + cc];
        T na = w[1][1], nb = w[1][2], nc = w[2][1], nd = w[2][2];
        if (!outside) {
            int xg = 0;
            if (EX) xg = (2 * m + 1 == glo) ? 1 : ((2 * m + 2 == ghi) ? 2 : 0);
            // columns entirely outside the domain only carry finite filler
            const bool xout = EX && (2 * m + 2 <= glo || 2 * m + 1 >= ghi);
            if (!xout) group_update(w, k, xg, yg, na, nb, nc, nd);
        }
        o[2 * m] = na; o[2 * m + 1] = nb;
        o[C + 2 * m] = nc; o[C + 2 * m + 1] = nd;
    }
}

template <typename T, int C, bool EX>
__device__ __forceinline__ void temporal2d_stage(const T (&P0)[C], const T (&P1)[C], const T (&Q0)[C],
                                                 const T (&Q1)[C], T (&N0)[C], T (&N1)[C],
                                                 const Coef2<T>& k, int glo, int ghi) {
    constexpr unsigned FULL = 0xffffffffu;
    const T r = k.r, g2 = k.g2, g4 = k.g4;
    T Ra[C / 2], Rb[C / 2 + 1], Rc[C / 2], Rd[C / 2 + 1];
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
    Rb[C / 2] = __shfl_down_sync(FULL, Rb[0], 1);
    Rd[C / 2] = __shfl_down_sync(FULL, Rd[0], 1);
#pragma unroll
    for (int m = 0; m < C / 2; ++m) {
        const T ra = Ra[m], rb = Rb[m + 1], rc = Rc[m], rd = Rd[m + 1];
        const T E1 = ra - rd, E2 = rb - rc;
        const T Q = (ra + rd) - (rb + rc);
        T na = fma(-g4, Q, fma(-g2, E1, ra));
        T nd = fma(-g4, Q, fma(g2, E1, rd));
        T nb = fma(g4, Q, fma(-g2, E2, rb));
        T nc = fma(g4, Q, fma(g2, E2, rc));
        if constexpr (EX) {
            if (2 * m + 1 == glo) {            // members a, c are the ghost column x = -1
                const T s = (rb - k.xlo) + (rd - k.xlo), df = rb - rd;
                nb = fma(-k.h3, df, fma(-k.h1, s, rb));
                nd = fma(k.h3, df, fma(-k.h1, s, rd));
                na = k.xlo; nc = k.xlo;
            } else if (2 * m + 2 == ghi) {     // members b, d are the ghost column x = nx
                const T s = (ra - k.xhi) + (rc - k.xhi), df = ra - rc;
                na = fma(-k.h3, df, fma(-k.h1, s, ra));
                nc = fma(k.h3, df, fma(-k.h1, s, rc));
                nb = k.xhi; nd = k.xhi;
            }
            // a ghost column inside a group that lies wholly outside the domain stays pinned
            if (2 * m + 2 == glo) { nb = k.xlo; nd = k.xlo; }
            if (2 * m + 1 == ghi) { na = k.xhi; nc = k.xhi; }
        }
        N0[2 * m] = na; N0[2 * m + 1] = nb;
        N1[2 * m] = nc; N1[2 * m + 1] = nd;
    }
}

// Row y of the lane's window (columns a0 .. a0+C-1) as loaded from HBM; rows and columns outside the
// grid return the Dirichlet value (ghost row/column) or a finite filler.  No shuffle here: the caller
// applies the `pre` shift when the data is consumed, so that the load stays in flight meanwhile.
template <typename T, int C, bool EX>
__device__ __forceinline__ void temporal2d_load_row(const T* __restrict__ uin, int nx, int ny,
                                                    const Coef2<T>& k, int y, int a0, T (&v)[C]) {
    constexpr int V = VecOf<T>::V;
    if ((unsigned)y < (unsigned)ny) {
        const T* __restrict__ row = uin + (int64_t)y * nx;
#pragma unroll
        for (int c = 0; c < C / V; ++c) {
            const int idx = a0 + c * V;
            T t[V];
            if (!EX || (idx >= 0 && idx + V <= nx)) {
                ld_vec(row + idx, t);
            } else {
#pragma unroll
                for (int j = 0; j < V; ++j) t[j] = (idx + j == -1) ? k.xlo : ((idx + j == nx) ? k.xhi : T(0));
            }
#pragma unroll
            for (int j = 0; j < V; ++j) v[c * V + j] = t[j];
        }
    } else {
        const T f = y == -1 ? k.ylo : (y == ny ? k.yhi : T(0));
#pragma unroll
        for (int j = 0; j < C; ++j) v[j] = f;
    }
}

template <typename T, int C, bool EX>
__device__ __forceinline__ void temporal2d_store_row(T* __restrict__ uout, int nx, int y, int o0,
                                                     int lane, int valid, int post, T (&v)[C]) {
    constexpr int V = VecOf<T>::V;
    for (int s = 0; s < post; ++s) shift_window<T, C>(v);
    T* __restrict__ row = uout + (int64_t)y * nx;
#pragma unroll
    for (int c = 0; c < C / V; ++c) {
        const int idx = o0 + c * V;
        if (lane * C + c * V < valid && idx + V <= nx) {
            T t[V];
#pragma unroll
            for (int j = 0; j < V; ++j) t[j] = v[c * V + j];
            st_vec(row + idx, t);
        }
    }
}

template <typename T, int C, int TB, bool EX>
__device__ __forceinline__ void temporal2d_strip(const T* __restrict__ uin, T* __restrict__ uout, int nx,
                                                 int ny, const Coef2<T>* __restrict__ coef,
                                                 const Temporal2dGeom g, int strip, int seg, int lane) {
    constexpr unsigned FULL = 0xffffffffu;
    const Coef2<T> k = *coef;
    const int a0 = strip * g.valid - g.shift + lane * C;     // column of slot 0 at load time
    const int o0 = strip * g.valid + lane * C;               // column of slot 0 at store time
    const int ys = g.ybase + 2 * g.hp * seg;                 // first output row
    const int ye = ys + 2 * g.hp < ny ? ys + 2 * g.hp : ny;
    const int Y0 = ys - TB;
    int glo = -(1 << 20), ghi = 1 << 20;     // window slots of the ghost columns at stage 0
    if constexpr (EX) {
        const int w0 = a0 + g.pre;
        const int dlo = -1 - w0, dhi = nx - w0;
        glo = dlo < -(1 << 20) ? -(1 << 20) : (dlo > (1 << 20) ? (1 << 20) : dlo);
        ghi = dhi < -(1 << 20) ? -(1 << 20) : (dhi > (1 << 20) ? (1 << 20) : dhi);
    }
    T prev[TB][2][C];
#pragma unroll
    for (int l = 0; l < TB; ++l)
#pragma unroll
        for (int j = 0; j < C; ++j) { prev[l][0][j] = T(0); prev[l][1][j] = T(0); }
    T cur[2][C], nxt[2][C];
    temporal2d_load_row<T, C, EX>(uin, nx, ny, k, Y0, a0, cur[0]);
    temporal2d_load_row<T, C, EX>(uin, nx, ny, k, Y0 + 1, a0, cur[1]);
    if (g.pre) { shift_window<T, C>(cur[0]); shift_window<T, C>(cur[1]); }
    const int iters = g.hp + TB;
#pragma unroll 1
    for (int it = 0; it < iters; ++it) {
        const int y0 = Y0 + 2 * it;
        // prefetch the next row pair; it is consumed (and pre-shifted) at the end of this iteration
        temporal2d_load_row<T, C, EX>(uin, nx, ny, k, y0 + 2, a0, nxt[0]);
        temporal2d_load_row<T, C, EX>(uin, nx, ny, k, y0 + 3, a0, nxt[1]);
#pragma unroll
        for (int l = 0; l < TB; ++l) {
            const int j = y0 - 1 - l;              // lower row of this stage's groups
            T nw[2][C];
            if ((unsigned)j < (unsigned)(ny - 1)) {            // rows j and j+1 both interior
                temporal2d_stage<T, C, EX>(prev[l][0], prev[l][1], cur[0], cur[1], nw[0], nw[1], k, glo - l, ghi - l);
            } else {
                T win[4][C + 2];
#pragma unroll
                for (int s = 0; s < C; ++s) {
                    win[0][s] = prev[l][0][s]; win[1][s] = prev[l][1][s];
                    win[2][s] = cur[0][s]; win[3][s] = cur[1][s];
                }
                win[0][C] = __shfl_down_sync(FULL, prev[l][0][0], 1); win[0][C + 1] = T(0);
                win[1][C] = __shfl_down_sync(FULL, prev[l][1][0], 1);
                win[1][C + 1] = __shfl_down_sync(FULL, prev[l][1][1], 1);
                win[2][C] = __shfl_down_sync(FULL, cur[0][0], 1);
                win[2][C + 1] = __shfl_down_sync(FULL, cur[0][1], 1);
                win[3][C] = __shfl_down_sync(FULL, cur[1][0], 1); win[3][C + 1] = T(0);
                T o[2][C];
                const int yg = j == -1 ? 1 : (j + 1 == ny ? 2 : 0);
                temporal2d_stage_edge<T, C, EX>(&win[0][0], &o[0][0], coef, glo - l, ghi - l, yg, yg == 0);
#pragma unroll
                for (int s = 0; s < C; ++s) { nw[0][s] = o[0][s]; nw[1][s] = o[1][s]; }
            }
#pragma unroll
            for (int s = 0; s < C; ++s) {
                prev[l][0][s] = cur[0][s]; prev[l][1][s] = cur[1][s];
                cur[0][s] = nw[0][s]; cur[1][s] = nw[1][s];
            }
        }
        // cur now holds level-TB rows (y0 - TB, y0 - TB + 1)
        if (it >= TB) {
            const int yo = y0 - TB;
            if (yo >= 0 && yo < ye)
                temporal2d_store_row<T, C, EX>(uout, nx, yo, o0, lane, g.valid, g.post, cur[0]);
            if (yo + 1 >= 0 && yo + 1 < ye)
                temporal2d_store_row<T, C, EX>(uout, nx, yo + 1, o0, lane, g.valid, g.post, cur[1]);
        }
#pragma unroll
        for (int s = 0; s < C; ++s) { cur[0][s] = nxt[0][s]; cur[1][s] = nxt[1][s]; }
        if (g.pre) { shift_window<T, C>(cur[0]); shift_window<T, C>(cur[1]); }
    }
}

template <typename T, int C, int TB>
__global__ void __launch_bounds__(kTemporal2dWarps * 32)
ge2d_temporal_kernel(const T* __restrict__ uin, T* __restrict__ uout, int nx, int ny,
                     const Coef2<T>* __restrict__ coef, const Temporal2dGeom g) {
    const int lane = threadIdx.x & 31;
    const int warp = threadIdx.x >> 5;
    const int strip = blockIdx.x * kTemporal2dWarps + warp;
    const int seg = blockIdx.y;
    if (strip >= g.strips) return;
    const int lo = strip * g.valid - g.shift;
    const bool ex = lo < 0 || lo + 32 * C > nx;
    if (ex) temporal2d_strip<T, C, TB, true>(uin, uout, nx, ny, coef, g, strip, seg, lane);
    else    temporal2d_strip<T, C, TB, false>(uin, uout, nx, ny, coef, g, strip, seg, lane);
}

// Host launcher: TB levels starting at a level of the given phase.  Requires nx % V == 0,
// 16-byte aligned buffers and nx, ny < 2^30 (32-bit row/column arithmetic in the kernel).
template <typename T, int C, int TB>
inline cudaError_t temporal2d_launch(const T* uin, T* uout, int64_t nx, int64_t ny, const Coef2<T>* coef,
                                     int phase, int hp, cudaStream_t s) {
    const Temporal2dGeom g = temporal2d_geom(C, VecOf<T>::V, TB, phase, nx, ny, hp);
    dim3 grid((unsigned)((g.strips + kTemporal2dWarps - 1) / kTemporal2dWarps), (unsigned)g.segs);
    ge2d_temporal_kernel<T, C, TB><<<grid, kTemporal2dWarps * 32, 0, s>>>(uin, uout, (int)nx, (int)ny, coef, g);
    return cudaGetLastError();
}

}  // namespace ge
