// ge_temporal_src.cuh -- strategy B in REGISTERS for non-constant problem data (DESIGN.md
// reading R-N3): a stationary source term tau*f and boundary values that move from level to level, two-point
// groups, batched rods.  The warp-per-tile, drift-free form of ge_temporal.cuh / ge_resident.cuh (levels in pairs
// R / L that slide the window right, then left; one shuffle per lane and level) with a second register array: lane
// t keeps tau*f of its window's C nodes and of the node right of it (the window reaches it in the shifted state).
//
// Arithmetic: the level code of ge_resident.cuh with the source added to every right-hand side exactly where
// ge_level_src.cuh adds it (p = fma(r, a - b, b) + s, the same rounding), so the results equal the per-level
// kernel's bit for bit.  Boundary values (bc = [batch][levels of the run + 1][2], as ge1d_window_kernel takes them):
// a level n -> n+1 reads the OLD value b[n] where a Dirichlet node is an out-of-group neighbour (levels I and L at
// the low end, level I at the high end -- level L finds the high ghost in the window, where level R left it) and
// the NEW value b[n+1] where it is the in-group partner (level R at both ends).
//
// ge1d_window_kernel (shared memory, any length and alignment) stays the general form; this kernel takes rows of
// whole aligned vectors that hold at least one tile.
#pragma once
#include "ge_common.cuh"
#include "ge_resident.cuh"
#include "ge_temporal.cuh"

namespace ge {

// R: even state -> shifted state (a phase-1 level); s[j] = tau*f of the node in slot j of the EVEN state, j = 0 .. C
template <typename T, int C, bool BC>
__device__ __forceinline__ void level_R_src(T (&v)[C], T& x0, const ResidentCtx<T, false>& c, const T (&s)[C + 1]) {
    const T r = c.r, g = c.g;
    T e = v[1] - v[0];
    T pprev = fma(-r, e, v[1]) + s[1];
    const T z0 = fma(r, e, v[0]) + s[0];
    const T zin = from_right<T, false>(c, z0, 0);
    if constexpr (BC) x0 = fma(-c.e, z0 - c.lo, z0);          // node 1, single: its partner node 0 at the new level
#pragma unroll
    for (int m = 1; m < C / 2; ++m) {
        e = v[2 * m + 1] - v[2 * m];
        const T pm = fma(-r, e, v[2 * m + 1]) + s[2 * m + 1];
        const T zm = fma(r, e, v[2 * m]) + s[2 * m];
        const T t = zm - pprev;
        v[2 * m - 2] = fma(g, t, pprev);
        v[2 * m - 1] = fma(-g, t, zm);
        pprev = pm;
    }
    const bool hi = BC && c.is_hi;
    const T ql = hi ? c.hi : zin;
    const T gl = hi ? c.e : g;
    const T t = ql - pprev;
    v[C - 2] = fma(gl, t, pprev);
    const T last = fma(-gl, t, ql);
    v[C - 1] = hi ? c.hi : last;                               // the ghost holds the new level's boundary value
}

// L: shifted state -> even state (a phase-0 level); slot j of the shifted state is the node of s[j + 1]
template <typename T, int C, bool BC>
__device__ __forceinline__ void level_L_src(T (&v)[C], const T x0, const ResidentCtx<T, false>& c, const T (&s)[C + 1]) {
    const T r = c.r, g = c.g;
    T e = v[C - 1] - v[C - 2];
    const T plast = fma(-r, e, v[C - 1]) + s[C];
    T znext = fma(r, e, v[C - 2]) + s[C - 1];
    const T pin = from_left<T, false>(c, plast, 0);
#pragma unroll
    for (int m = C / 2 - 2; m >= 0; --m) {
        e = v[2 * m + 1] - v[2 * m];
        const T pm = fma(-r, e, v[2 * m + 1]) + s[2 * m + 2];
        const T zm = fma(r, e, v[2 * m]) + s[2 * m + 1];
        const T t = znext - pm;
        v[2 * m + 2] = fma(g, t, pm);
        v[2 * m + 3] = fma(-g, t, znext);
        znext = zm;
    }
    T P = pin;
    if constexpr (BC) {
        const T pl = fma(-r, x0 - c.lo, x0) + s[0];            // pair (1,2): node 0 at the OLD level is its left neighbour
        P = c.is_lo ? pl : pin;
    }
    const T t = znext - P;
    v[0] = fma(g, t, P);
    v[1] = fma(-g, t, znext);
}

// I: even state -> even state, pairs inside the lane (a phase-0 level)
template <typename T, int C, bool BC>
__device__ __forceinline__ void level_I_src(T (&v)[C], const ResidentCtx<T, false>& c, const T (&s)[C + 1]) {
    const T r = c.r, g = c.g;
    T a = from_left<T, false>(c, v[C - 1], 0);
    T d = from_right<T, false>(c, v[0], 0);
    if (BC && c.is_lo) a = c.lo;
    if (BC && c.is_hi) d = c.hi;
#pragma unroll
    for (int m = 0; m < C / 2; ++m) {
        const T b = v[2 * m], cc = v[2 * m + 1];
        const T dd = (m == C / 2 - 1) ? d : v[2 * m + 2];
        const T p = fma(r, a - b, b) + s[2 * m];
        const T q = fma(r, dd - cc, cc) + s[2 * m + 1];
        const T t = q - p;
        a = cc;
        v[2 * m] = fma(g, t, p);
        v[2 * m + 1] = fma(-g, t, q);
    }
}

// One tile: g.tb levels from a level of phase (g.pre ? 0 : 1).  bcr: the rod's boundary values, [level][lo, hi],
// bcr[0..1] = at the launch's first level.
template <typename T, int C, bool BC>
__device__ __forceinline__ void temporal1d_tile_src(const T* __restrict__ in, T* __restrict__ out, const T* __restrict__ src,
                                                    const T* __restrict__ bcr, int64_t nx, const Coef1<T>& k,
                                                    const Temporal1dGeom g, int64_t a0, int64_t out_lo, int64_t out_hi,
                                                    bool first, bool last, int lane) {
    constexpr int V = VecOf<T>::V;
    const int64_t e0 = a0 + (int64_t)lane * C;
    T v[C], s[C + 1];
#pragma unroll
    for (int c = 0; c < C / V; ++c) {
        T t[V];
        ld_vec(in + e0 + c * V, t);
#pragma unroll
        for (int j = 0; j < V; ++j) v[c * V + j] = t[j];
        if (src) ld_vec(src + e0 + c * V, t);
#pragma unroll
        for (int j = 0; j < V; ++j) s[c * V + j] = src ? t[j] : T(0);
    }
    {   // the node right of the lane's window: the next lane's first, or the next tile's
        T nxt = __shfl_down_sync(0xffffffffu, s[0], 1);
        if (lane == 31) nxt = (src && e0 + C < nx) ? __ldg(src + e0 + C) : T(0);
        s[C] = nxt;
    }
    ResidentCtx<T, false> cx;
    cx.r = k.r; cx.g = k.g; cx.e = k.e; cx.lo = k.lo; cx.hi = k.hi;
    cx.is_lo = BC && first && lane == 0; cx.is_hi = BC && last && lane == 31;
    cx.lane = lane; cx.warp = 0; cx.nwarps = 1; cx.sx = nullptr;
    T x0 = T(0);
    int left = g.tb, lev = 0;
    if (g.pre) {
        if constexpr (BC) { cx.lo = bcr[2 * lev]; cx.hi = bcr[2 * lev + 1]; }
        level_I_src<T, C, BC>(v, cx, s);
        --left; ++lev;
    }
#pragma unroll 1
    for (; left >= 2; left -= 2, lev += 2) {
        if constexpr (BC) { cx.lo = bcr[2 * (lev + 1)]; cx.hi = bcr[2 * (lev + 1) + 1]; }     // R: new values
        level_R_src<T, C, BC>(v, x0, cx, s);
        if constexpr (BC) cx.lo = bcr[2 * (lev + 1)];                                         // L: old value = R's new
        level_L_src<T, C, BC>(v, x0, cx, s);
    }
    if (left) {
        if constexpr (BC) { cx.lo = bcr[2 * (lev + 1)]; cx.hi = bcr[2 * (lev + 1) + 1]; }
        level_R_src<T, C, BC>(v, x0, cx, s);
        unshift<T, C, false, BC>(v, x0, cx, 0);
    }
#pragma unroll
    for (int c = 0; c < C / V; ++c) {
        const int64_t e = e0 + c * V;
        if (e >= out_lo && e < out_hi) {
            T t[V];
#pragma unroll
            for (int j = 0; j < V; ++j) t[j] = v[c * V + j];
            st_vec(out + e, t);
        }
    }
}

template <typename T, int C>
__global__ void __launch_bounds__(kTemporalWarps * 32)
ge1d_temporal_src_kernel(const T* __restrict__ uin, T* __restrict__ uout, const T* __restrict__ src, const T* __restrict__ bc,
                         int64_t bc_lev, int64_t bc_stride, int64_t nx, int64_t batch, const Coef1<T>* __restrict__ coef,
                         const Temporal1dGeom g, const Temporal1dTiles tl) {
    const int lane = threadIdx.x & 31;
    const int warp = threadIdx.x >> 5;
    const int64_t tile = (int64_t)blockIdx.x * kTemporalWarps + warp;
    if (tile >= tl.ntiles) return;
    const bool first = tile == 0, last = tile == tl.nreg;
    const int64_t a0 = first ? 0 : (last ? nx - 32 * (int64_t)C : tile * g.valid - g.halo);
    const int64_t out_lo = tile * g.valid;
    const int64_t out_hi = last ? nx : out_lo + g.valid;
    for (int64_t rod = blockIdx.y; rod < batch; rod += gridDim.y) {
        const Coef1<T> k = coef[rod];
        const T* __restrict__ in = uin + rod * nx;
        T* __restrict__ out = uout + rod * nx;
        const T* __restrict__ sr = src ? src + rod * nx : nullptr;
        const T* __restrict__ bcr = bc + (rod * bc_stride + bc_lev) * 2;
        if (first || last) temporal1d_tile_src<T, C, true>(in, out, sr, bcr, nx, k, g, a0, out_lo, out_hi, first, last, lane);
        else               temporal1d_tile_src<T, C, false>(in, out, sr, bcr, nx, k, g, a0, out_lo, out_hi, false, false, lane);
    }
}

// Requires nx % V == 0, nx >= 32*C, 16-byte aligned rows of u and of src, 1 <= tb <= temporal1d_max_tb(C).
template <typename T, int C>
inline cudaError_t temporal1d_src_launch(const T* uin, T* uout, const T* src, const T* bc, int64_t bc_lev, int64_t bc_stride,
                                         int64_t nx, int64_t batch, const Coef1<T>* coef, int tb, int phase, cudaStream_t s) {
    const Temporal1dGeom g = temporal1d_geom(C, VecOf<T>::V, tb, phase);
    const Temporal1dTiles tl = temporal1d_tiles(C, g, nx);
    dim3 grid((unsigned)((tl.ntiles + kTemporalWarps - 1) / kTemporalWarps), (unsigned)(batch < 65535 ? batch : 65535));
    ge1d_temporal_src_kernel<T, C><<<grid, kTemporalWarps * 32, 0, s>>>(uin, uout, src, bc, bc_lev, bc_stride, nx, batch, coef, g, tl);
    return cudaGetLastError();
}

// ---------------------------------------------------------------- variable diffusivity (reading R-VAR) ------
// One number per link, rl[j] = link between nodes j and j+1 (ge_level_var.cuh).  A lane whose even-state window
// holds the nodes n0 .. n0+C-1 keeps the C + 1 links lk[j] = rl[n0 + j], j = -1 .. C-1 (L[j + 1]; lk[j] joins the
// nodes of slots j and j+1), and the pair factors g = rm / (1 + 2 rm) of the C links inside its window's reach:
// gE[m] of lk[2m] (the pairs of a phase-0 level), gO[m] of lk[2m+1] (phase 1) -- one division per link and launch
// instead of one per pair and level.  The shared difference e across an out-of-group link serves both adjacent pairs
// as in the constant-coefficient code, with that link's number: p = b - lk e, z = a + lk e (the per-level kernel's
// fma(rl, a - b, b), same rounding).
template <typename T, int C>
struct VarLinks { T L[C + 1]; T gE[C / 2]; T gO[C / 2]; };

template <typename T, int C, bool BC>
__device__ __forceinline__ void level_R_var(T (&v)[C], T& x0, const ResidentCtx<T, false>& c, const VarLinks<T, C>& k) {
    T e = v[1] - v[0];
    T pprev = fma(-k.L[1], e, v[1]);
    const T z0 = fma(k.L[1], e, v[0]);
    const T zin = from_right<T, false>(c, z0, 0);
    if constexpr (BC) {                                        // node 1, single: link (0, 1), cut pair
        const T ge = k.L[0] / (T(1) + k.L[0]);
        x0 = fma(-ge, z0 - c.lo, z0);
    }
#pragma unroll
    for (int m = 1; m < C / 2; ++m) {
        e = v[2 * m + 1] - v[2 * m];
        const T pm = fma(-k.L[2 * m + 1], e, v[2 * m + 1]);
        const T zm = fma(k.L[2 * m + 1], e, v[2 * m]);
        const T t = zm - pprev;                                // pair (slots 2m-1, 2m): inner link lk[2m-1]
        v[2 * m - 2] = fma(k.gO[m - 1], t, pprev);
        v[2 * m - 1] = fma(-k.gO[m - 1], t, zm);
        pprev = pm;
    }
    const bool hi = BC && c.is_hi;
    const T ql = hi ? c.hi : zin;
    T gl = k.gO[C / 2 - 1];                                    // pair (slot C-1, next lane's slot 0): inner link lk[C-1]
    if constexpr (BC) { if (hi) gl = k.L[C] / (T(1) + k.L[C]); }
    const T t = ql - pprev;
    v[C - 2] = fma(gl, t, pprev);
    const T last = fma(-gl, t, ql);
    v[C - 1] = hi ? c.hi : last;
}

template <typename T, int C, bool BC>
__device__ __forceinline__ void level_L_var(T (&v)[C], const T x0, const ResidentCtx<T, false>& c, const VarLinks<T, C>& k) {
    // shifted state: slot j holds the node of even slot j + 1; slots j, j+1 are joined by lk[j + 1]
    T e = v[C - 1] - v[C - 2];
    const T plast = fma(-k.L[C], e, v[C - 1]);
    T znext = fma(k.L[C], e, v[C - 2]);
    const T pin = from_left<T, false>(c, plast, 0);
#pragma unroll
    for (int m = C / 2 - 2; m >= 0; --m) {
        e = v[2 * m + 1] - v[2 * m];                           // across lk[2m+1]
        const T pm = fma(-k.L[2 * m + 2], e, v[2 * m + 1]);
        const T zm = fma(k.L[2 * m + 2], e, v[2 * m]);
        const T t = znext - pm;                                // pair (even slots 2m+2, 2m+3): inner link lk[2m+2]
        v[2 * m + 2] = fma(k.gE[m + 1], t, pm);
        v[2 * m + 3] = fma(-k.gE[m + 1], t, znext);
        znext = zm;
    }
    T P = pin;
    if constexpr (BC) {
        const T pl = fma(-k.L[0], x0 - c.lo, x0);              // pair (1,2): outer link (0, 1)
        P = c.is_lo ? pl : pin;
    }
    const T t = znext - P;                                     // pair (even slots 0, 1): inner link lk[0]
    v[0] = fma(k.gE[0], t, P);
    v[1] = fma(-k.gE[0], t, znext);
}

template <typename T, int C, bool BC>
__device__ __forceinline__ void level_I_var(T (&v)[C], const ResidentCtx<T, false>& c, const VarLinks<T, C>& k) {
    T a = from_left<T, false>(c, v[C - 1], 0);
    T d = from_right<T, false>(c, v[0], 0);
    if (BC && c.is_lo) a = c.lo;
    if (BC && c.is_hi) d = c.hi;
#pragma unroll
    for (int m = 0; m < C / 2; ++m) {
        const T b = v[2 * m], cc = v[2 * m + 1];
        const T dd = (m == C / 2 - 1) ? d : v[2 * m + 2];
        const T p = fma(k.L[2 * m], a - b, b);                 // outer links lk[2m-1], lk[2m+1]; inner lk[2m]
        const T q = fma(k.L[2 * m + 2], dd - cc, cc);
        const T t = q - p;
        a = cc;
        v[2 * m] = fma(k.gE[m], t, p);
        v[2 * m + 1] = fma(-k.gE[m], t, q);
    }
}

// rl: the rod's link numbers, nx + 1 of them (any alignment: rows of nx + 1 elements)
template <typename T, int C, bool BC>
__device__ __forceinline__ void temporal1d_tile_var(const T* __restrict__ in, T* __restrict__ out, const T* __restrict__ rl,
                                                    const Coef1<T>& kc, const Temporal1dGeom g, int64_t a0,
                                                    int64_t out_lo, int64_t out_hi, bool first, bool last, int lane) {
    constexpr int V = VecOf<T>::V;
    const int64_t e0 = a0 + (int64_t)lane * C;                 // element of slot 0 = node e0 + 1
    T v[C];
#pragma unroll
    for (int c = 0; c < C / V; ++c) {
        T t[V];
        ld_vec(in + e0 + c * V, t);
#pragma unroll
        for (int j = 0; j < V; ++j) v[c * V + j] = t[j];
    }
    VarLinks<T, C> k;
#pragma unroll
    for (int j = 0; j <= C; ++j) k.L[j] = __ldg(rl + e0 + j);  // lk[j-1] = rl[n0 + j - 1], n0 = e0 + 1
#pragma unroll
    for (int m = 0; m < C / 2; ++m) {
        k.gE[m] = k.L[2 * m + 1] / fma(T(2), k.L[2 * m + 1], T(1));
        k.gO[m] = k.L[2 * m + 2] / fma(T(2), k.L[2 * m + 2], T(1));
    }
    ResidentCtx<T, false> cx;
    cx.r = kc.r; cx.g = kc.g; cx.e = kc.e; cx.lo = kc.lo; cx.hi = kc.hi;
    cx.is_lo = BC && first && lane == 0; cx.is_hi = BC && last && lane == 31;
    cx.lane = lane; cx.warp = 0; cx.nwarps = 1; cx.sx = nullptr;
    T x0 = T(0);
    int left = g.tb;
    if (g.pre) { level_I_var<T, C, BC>(v, cx, k); --left; }
#pragma unroll 1
    for (; left >= 2; left -= 2) {
        level_R_var<T, C, BC>(v, x0, cx, k);
        level_L_var<T, C, BC>(v, x0, cx, k);
    }
    if (left) {
        level_R_var<T, C, BC>(v, x0, cx, k);
        unshift<T, C, false, BC>(v, x0, cx, 0);
    }
#pragma unroll
    for (int c = 0; c < C / V; ++c) {
        const int64_t e = e0 + c * V;
        if (e >= out_lo && e < out_hi) {
            T t[V];
#pragma unroll
            for (int j = 0; j < V; ++j) t[j] = v[c * V + j];
            st_vec(out + e, t);
        }
    }
}

template <typename T, int C>
__global__ void __launch_bounds__(kTemporalWarps * 32)
ge1d_temporal_var_kernel(const T* __restrict__ uin, T* __restrict__ uout, const T* __restrict__ rl, int64_t nx, int64_t batch,
                         const Coef1<T>* __restrict__ coef, const Temporal1dGeom g, const Temporal1dTiles tl) {
    const int lane = threadIdx.x & 31;
    const int warp = threadIdx.x >> 5;
    const int64_t tile = (int64_t)blockIdx.x * kTemporalWarps + warp;
    if (tile >= tl.ntiles) return;
    const bool first = tile == 0, last = tile == tl.nreg;
    const int64_t a0 = first ? 0 : (last ? nx - 32 * (int64_t)C : tile * g.valid - g.halo);
    const int64_t out_lo = tile * g.valid;
    const int64_t out_hi = last ? nx : out_lo + g.valid;
    for (int64_t rod = blockIdx.y; rod < batch; rod += gridDim.y) {
        const Coef1<T> k = coef[rod];
        const T* __restrict__ in = uin + rod * nx;
        T* __restrict__ out = uout + rod * nx;
        const T* __restrict__ lr = rl + rod * (nx + 1);
        if (first || last) temporal1d_tile_var<T, C, true>(in, out, lr, k, g, a0, out_lo, out_hi, first, last, lane);
        else               temporal1d_tile_var<T, C, false>(in, out, lr, k, g, a0, out_lo, out_hi, false, false, lane);
    }
}

// Requires nx % V == 0, nx >= 32*C, 16-byte aligned rows of u, 1 <= tb <= temporal1d_max_tb(C).
template <typename T, int C>
inline cudaError_t temporal1d_var_launch(const T* uin, T* uout, const T* rl, int64_t nx, int64_t batch, const Coef1<T>* coef,
                                         int tb, int phase, cudaStream_t s) {
    const Temporal1dGeom g = temporal1d_geom(C, VecOf<T>::V, tb, phase);
    const Temporal1dTiles tl = temporal1d_tiles(C, g, nx);
    dim3 grid((unsigned)((tl.ntiles + kTemporalWarps - 1) / kTemporalWarps), (unsigned)(batch < 65535 ? batch : 65535));
    ge1d_temporal_var_kernel<T, C><<<grid, kTemporalWarps * 32, 0, s>>>(uin, uout, rl, nx, batch, coef, g, tl);
    return cudaGetLastError();
}

}  // namespace ge
