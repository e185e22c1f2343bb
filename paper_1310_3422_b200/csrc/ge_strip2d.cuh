// ge_strip2d.cuh -- strategy B (2-D), drift-free: TB levels per HBM round trip,
// state in registers and lane-private shared memory, no barrier.
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
//   * the previous row pair of every stage lives in lane-private SHARED memory
//     slots (conflict-free 16-byte accesses, no synchronisation), so registers
//     hold only the pair that flows through the stages: 20+ warps per SM, no
//     rotating register moves.  Row pairs arrive through a cp.async ring in
//     shared memory, requested two iterations ahead.
//   * groups cut by a y edge (and rows outside the grid) take a generic
//     out-of-line path built on ge_level.cuh group_update.
// Arithmetic: 6.75 flop-instructions per node update, the expression tree of
// ge2d_level_kernel (bit-identical results).
#pragma once
#include "ge_common.cuh"
#include "ge_level.cuh"

namespace ge {

#ifndef GE_STRIP_WARPS
#define GE_STRIP_WARPS 4
#endif
#ifndef GE_STRIP_RING
#define GE_STRIP_RING 3
#endif
constexpr int kStripWarps = GE_STRIP_WARPS;   // warps per CTA = adjacent strips (their halos share L2 lines)

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
    // cooperative strips (COOP > 1 warps share one strip; see strip_neighbour)
    int warp;              // warp of the strip, 0 .. COOP-1
    int gl;                // lane of the strip, warp*32 + lane
    T* xch;                // shared memory: exchange lines of the strip
    T* xslow;              // shared memory: [COOP*32 lanes][4 values] for the y-edge path
};

// ---- cooperative strips ----------------------------------------------------------------------------
// COOP adjacent warps of a CTA own ONE strip of COOP*32*C columns and march through the same row pairs in
// step.  A stage needs from the neighbouring LANE two right-hand sides (R stages: of the lane to the right,
// L stages: to the left).  Inside a warp that is a pair of shuffles; with COOP > 1 every lane publishes its
// two values in a shared-memory line of the strip and reads its neighbour's, so that the last (first) lane
// of a warp gets them from the next (previous) WARP instead of recomputing TB stale columns: only the two
// ends of the CTA's strip carry a redundant halo.  Ordering between two adjacent warps is a pair of named
// barriers (bar.arrive by the producer, bar.sync by the consumer, 64 threads): barrier 1+w orders "warp w+1
// published, warp w may read" (R stages), barrier COOP+w "warp w published, warp w+1 may read" (L stages).
// A producer never waits; since R and L stages alternate, a warp can run at most one stage ahead of its
// neighbour, which is also why one line per stage type (and iteration parity, for slack) is enough: the
// producer of an R line rewrites it two stages later, after an L stage that needed the consumer's arrive,
// which follows the consumer's read in program order.
__device__ __forceinline__ void bar_arrive(int id, int n) { asm volatile("bar.arrive %0, %1;" ::"r"(id), "r"(n) : "memory"); }
__device__ __forceinline__ void bar_sync(int id, int n) { asm volatile("bar.sync %0, %1;" ::"r"(id), "r"(n) : "memory"); }

// elements of the exchange area of one strip: [2 stage types][2 iteration parities] lines of [COOP*32 lanes]
// [2 values], then the line of the y-edge path [COOP*32 lanes][4 values]
template <int COOP> struct StripXch {
    static constexpr int lines = COOP > 1 ? 4 * COOP * 32 * 2 : 0;
    static constexpr int elems = COOP > 1 ? lines + COOP * 32 * 4 : 0;
};

// RIGHT: the values (a, b) of lane gl+1, else of lane gl-1.  The lanes at the two ends of the strip get
// their own values back (stale columns of the CTA's halo, as lane 31 / lane 0 of a lone warp do).
template <typename T, int COOP, bool RIGHT>
__device__ __forceinline__ void strip_neighbour(T a, T b, T& na, T& nb, const Strip2dCtx<T>& k, int par) {
    constexpr unsigned FULL = 0xffffffffu;
    if constexpr (COOP == 1) {
        na = RIGHT ? __shfl_down_sync(FULL, a, 1) : __shfl_up_sync(FULL, a, 1);
        nb = RIGHT ? __shfl_down_sync(FULL, b, 1) : __shfl_up_sync(FULL, b, 1);
    } else {
        T* line = k.xch + ((RIGHT ? 0 : 2) + par) * (COOP * 32 * 2);
        if constexpr (sizeof(T) == 4) *reinterpret_cast<float2*>(line + 2 * k.gl) = make_float2(a, b);
        else                          *reinterpret_cast<double2*>(line + 2 * k.gl) = make_double2(a, b);
        if constexpr (RIGHT) {
            if (k.warp > 0) bar_arrive(1 + k.warp - 1, 64);
            if (k.warp < COOP - 1) bar_sync(1 + k.warp, 64); else __syncwarp();
        } else {
            if (k.warp < COOP - 1) bar_arrive(COOP + k.warp, 64);
            if (k.warp > 0) bar_sync(COOP + k.warp - 1, 64); else __syncwarp();
        }
        int nl = RIGHT ? k.gl + 1 : k.gl - 1;
        nl = nl < 0 ? 0 : (nl > COOP * 32 - 1 ? COOP * 32 - 1 : nl);
        if constexpr (sizeof(T) == 4) { const float2 v = *reinterpret_cast<const float2*>(line + 2 * nl); na = v.x; nb = v.y; }
        else                          { const double2 v = *reinterpret_cast<const double2*>(line + 2 * nl); na = v.x; nb = v.y; }
    }
}

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

// Right-hand sides a row pair X = (X0, X1) contributes to the columns in slots 2m (right members b, d
// of the group to the left) and 2m+1 (left members a, c).  The pair is the UPPER half of the group row
// (j, j+1) = (previous pair's row 1, X0): Rd[m], Rc[m] (members d, c in row X0, X1 the row above) --
// and, one iteration later, the LOWER half of the group row (X1, next pair's row 0): H[2m] = Rb[m],
// H[2m+1] = Ra[m] (members b, a in row X1, X0 the row below).  Both halves read nothing but this pair,
// so they are formed together when the pair passes (the y differences are shared) and only H -- one
// value per column instead of the two rows -- waits in the stage's state slot for the next pair.
template <typename T, int C>
__device__ __forceinline__ void strip_rhs_pair(const T (&X0)[C], const T (&X1)[C], T r, T (&H)[C],
                                               T (&Rc)[C / 2], T (&Rd)[C / 2]) {
#pragma unroll
    for (int m = 0; m < C / 2; ++m) {
        const T ex1 = X1[2 * m + 1] - X1[2 * m];
        const T ex0 = X0[2 * m + 1] - X0[2 * m];
        const T eyb = X1[2 * m] - X0[2 * m], eya = X1[2 * m + 1] - X0[2 * m + 1];
        H[2 * m] = fma(r, ex1 - eyb, X1[2 * m]);              // Rb: right + below
        H[2 * m + 1] = fma(-r, ex1 + eya, X1[2 * m + 1]);     // Ra: left + below
        Rd[m] = fma(r, ex0 + eyb, X0[2 * m]);                 // right + above
        Rc[m] = fma(r, eya - ex0, X0[2 * m + 1]);             // left + above
    }
}

// R: unshifted rows -> rows shifted right by one column.  H: lower-half right-hand sides left by the
// previous pair, Rc / Rd: upper half from the current pair.  N0 / N1 are the new rows of the group row;
// nx0[0..1]: new column 0 of those rows (lane is_lo only).
template <typename T, int C, bool BC>
__device__ __forceinline__ void strip_stage_R_given(const T (&H)[C], const T (&Rc)[C / 2], const T (&Rd)[C / 2],
                                                    T (&N0)[C], T (&N1)[C], T (&nx0)[2], const Strip2dCtx<T>& k,
                                                    const T RbN, const T RdN) {
#pragma unroll
    for (int m = 0; m < C / 2; ++m) {
        const T ra = H[2 * m + 1];
        const T rb = m + 1 < C / 2 ? H[2 * m + 2 < C ? 2 * m + 2 : 0] : RbN;
        const T rd = m + 1 < C / 2 ? Rd[m + 1 < C / 2 ? m + 1 : 0] : RdN;
        T na, nb, nc, nd;
        solve4(ra, rb, Rc[m], rd, k.g2, k.g4, na, nb, nc, nd);
        if constexpr (BC) {
            if (m == C / 2 - 1 && k.is_hi) {       // members b, d are the boundary column x = nx
                solve2(ra, Rc[m], k.xhi, k.h1, k.h3, na, nc);
                nb = k.xhi; nd = k.xhi;
            }
        }
        N0[2 * m] = na; N0[2 * m + 1] = nb;
        N1[2 * m] = nc; N1[2 * m + 1] = nd;
    }
    if constexpr (BC) solve2(H[0], Rd[0], k.xlo, k.h1, k.h3, nx0[0], nx0[1]);   // group (x = -1, 0)
}
template <typename T, int C, bool BC, int COOP = 1>
__device__ __forceinline__ void strip_stage_R(const T (&H)[C], const T (&Rc)[C / 2], const T (&Rd)[C / 2],
                                              T (&N0)[C], T (&N1)[C], T (&nx0)[2], const Strip2dCtx<T>& k, int par = 0) {
    T RbN, RdN;
    strip_neighbour<T, COOP, true>(H[0], Rd[0], RbN, RdN, k, par);
    strip_stage_R_given<T, C, BC>(H, Rc, Rd, N0, N1, nx0, k, RbN, RdN);
}

// L: rows shifted right by one column -> unshifted rows.  pP / pQ: column 0 of the previous pair's /
// the current pair's rows (lane is_lo only).
template <typename T, int C, bool BC>
__device__ __forceinline__ void strip_stage_L_given(const T (&H)[C], const T (&Rc)[C / 2], const T (&Rd)[C / 2],
                                                    const T (&pP)[2], const T (&pQ)[2],
                                                    T (&N0)[C], T (&N1)[C], const Strip2dCtx<T>& k, T ra, T rc) {
    if constexpr (BC) {
        if (k.is_lo) {     // members a, c are column 0; their left neighbour is the boundary column
            const T a = pP[1], c = pQ[0];
            ra = fma(-k.r, (a - k.xlo) + (a - pP[0]), a);
            rc = fma(k.r, (pQ[1] - c) - (c - k.xlo), c);
        }
    }
    solve4(ra, H[0], rc, Rd[0], k.g2, k.g4, N0[0], N0[1], N1[0], N1[1]);
#pragma unroll
    for (int m = 0; m + 1 < C / 2; ++m)
        solve4(H[2 * m + 1], H[2 * m + 2], Rc[m], Rd[m + 1], k.g2, k.g4, N0[2 * m + 2], N0[2 * m + 3],
               N1[2 * m + 2], N1[2 * m + 3]);
}
template <typename T, int C, bool BC, int COOP = 1>
__device__ __forceinline__ void strip_stage_L(const T (&H)[C], const T (&Rc)[C / 2], const T (&Rd)[C / 2],
                                              const T (&pP)[2], const T (&pQ)[2],
                                              T (&N0)[C], T (&N1)[C], const Strip2dCtx<T>& k, int par = 0) {
    T ra, rc;
    strip_neighbour<T, COOP, false>(H[C - 1], Rc[C / 2 - 1], ra, rc, k, par);
    strip_stage_L_given<T, C, BC>(H, Rc, Rd, pP, pQ, N0, N1, k, ra, rc);
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

// Out-of-line wrapper: io holds the four input rows P0, P1, Q0, Q1 (4*C values) followed by their
// column-0 values (4: lane is_lo, shifted rows); builds the extended rows (two neighbour columns
// per side, by shuffles), runs the generic stage and leaves N0, N1 (2*C values) and the new
// column 0 of the two rows (2) at the start of io.  Called from a warp-uniform branch.
template <typename T, int C, bool SHIFTED, int COOP = 1>
__device__ __noinline__ void strip_stage_slow(T* __restrict__ io, const Coef2<T>* __restrict__ coef, int yg,
                                              bool outside, bool is_lo, bool is_hi, T* __restrict__ xch = nullptr,
                                              int gl = 0) {
    constexpr unsigned FULL = 0xffffffffu;
    constexpr int E = C + 4;
    const T xlo = coef->xlo, xhi = coef->xhi;
    T ext[4 * E];
#pragma unroll
    for (int rr = 0; rr < 4; ++rr) {
        const T* v = io + rr * C;
#pragma unroll
        for (int s = 0; s < C; ++s) ext[rr * E + s + 2] = v[s];
        T l2, l1, r0, r1;
        if constexpr (COOP == 1) {
            l2 = __shfl_up_sync(FULL, v[C - 2], 1); l1 = __shfl_up_sync(FULL, v[C - 1], 1);
            r0 = __shfl_down_sync(FULL, v[0], 1); r1 = __shfl_down_sync(FULL, v[1], 1);
        } else {
            // the whole CTA (= the strip's COOP warps) is here: the edge test is the same for all of them
            T* sl = xch;            // the strip's y-edge line
            __syncthreads();
            sl[4 * gl] = v[0]; sl[4 * gl + 1] = v[1]; sl[4 * gl + 2] = v[C - 2]; sl[4 * gl + 3] = v[C - 1];
            __syncthreads();
            const int nl = gl > 0 ? gl - 1 : 0, nr = gl < COOP * 32 - 1 ? gl + 1 : gl;
            l2 = sl[4 * nl + 2]; l1 = sl[4 * nl + 3]; r0 = sl[4 * nr]; r1 = sl[4 * nr + 1];
        }
        if (is_lo) {
            if (SHIFTED) { l1 = io[4 * C + rr]; l2 = xlo; } else { l1 = xlo; l2 = T(0); }
        }
        if (is_hi) {
            if (SHIFTED) { r0 = T(0); r1 = T(0); } else { r0 = xhi; r1 = T(0); }
        }
        ext[rr * E + 0] = l2; ext[rr * E + 1] = l1;
        ext[rr * E + C + 2] = r0; ext[rr * E + C + 3] = r1;
    }
    T o[2 * C + 2];
    o[2 * C] = T(0); o[2 * C + 1] = T(0);
    strip_stage_edge<T, C, SHIFTED>(ext, o, coef, yg, outside, is_lo, is_hi);
#pragma unroll
    for (int s = 0; s < 2 * C + 2; ++s) io[s] = o[s];
}

// One EDGE stage-iteration (group rows j, j+1 not both interior): P = previous row pair of level l (with
// its column 0: xP), Q = current one, both raw; writes the level-(l+1) pair into N (xN).  Odd stages are
// L, even stages R.
template <typename T, int C, bool BC, int COOP = 1>
__device__ __forceinline__ void strip_stage_rows(const bool odd, const T (&P)[2][C], const T (&xP)[2],
                                                 const T (&Q)[2][C], const T (&xQ)[2], T (&N)[2][C], T (&xN)[2],
                                                 const Strip2dCtx<T>& k, const Coef2<T>* __restrict__ coef, int j,
                                                 int ny) {
    T io[4 * C + 4];
#pragma unroll
    for (int s = 0; s < C; ++s) {
        io[s] = P[0][s]; io[C + s] = P[1][s]; io[2 * C + s] = Q[0][s]; io[3 * C + s] = Q[1][s];
    }
    io[4 * C] = xP[0]; io[4 * C + 1] = xP[1]; io[4 * C + 2] = xQ[0]; io[4 * C + 3] = xQ[1];
    const int yg = j == -1 ? 1 : (j + 1 == ny ? 2 : 0);
    if (odd) strip_stage_slow<T, C, true, COOP>(io, coef, yg, yg == 0, BC && k.is_lo, BC && k.is_hi, k.xslow, k.gl);
    else     strip_stage_slow<T, C, false, COOP>(io, coef, yg, yg == 0, BC && k.is_lo, BC && k.is_hi, k.xslow, k.gl);
#pragma unroll
    for (int s = 0; s < C; ++s) { N[0][s] = io[s]; N[1][s] = io[C + s]; }
    if (!odd) { xN[0] = io[2 * C]; xN[1] = io[2 * C + 1]; }
}

// The pipeline state of every level 0 .. TB-1 lives in SHARED memory, in lane-private slots (vector c of
// lane t at [(c*32 + t)*V], conflict-free, no synchronisation).  What a stage keeps between two iterations
// is what the previous pair contributes to the next group row: its lower-half right-hand sides H (one value
// per column, strip_rhs_pair) -- or, when the next group row touches a y edge and takes the generic path,
// the raw pair (two rows; the same slot, the choice is warp-uniform and both sides derive it from j).
// Registers hold only the pair that flows through the stages, so 12+ warps fit on an SM and nothing
// rotates through register moves; shared-memory traffic per stage-iteration is one row in, one row out.
template <typename T, int C>
__device__ __forceinline__ void strip_lds(const T* __restrict__ sp, int lane, T (&v)[2][C]) {
    constexpr int V = VecOf<T>::V;
    using VT = typename VecOf<T>::type;
#pragma unroll
    for (int rr = 0; rr < 2; ++rr)
#pragma unroll
        for (int c = 0; c < C / V; ++c) {
            const VT q = *reinterpret_cast<const VT*>(sp + ((rr * (C / V) + c) * 32 + lane) * V);
            if constexpr (V == 4) { v[rr][c * V] = q.x; v[rr][c * V + 1] = q.y; v[rr][c * V + 2] = q.z; v[rr][c * V + 3] = q.w; }
            else { v[rr][c * V] = q.x; v[rr][c * V + 1] = q.y; }
        }
}
template <typename T, int C>
__device__ __forceinline__ void strip_sts(T* __restrict__ sp, int lane, const T (&v)[2][C]) {
    constexpr int V = VecOf<T>::V;
    using VT = typename VecOf<T>::type;
#pragma unroll
    for (int rr = 0; rr < 2; ++rr)
#pragma unroll
        for (int c = 0; c < C / V; ++c) {
            VT q;
            if constexpr (V == 4) { q.x = v[rr][c * V]; q.y = v[rr][c * V + 1]; q.z = v[rr][c * V + 2]; q.w = v[rr][c * V + 3]; }
            else { q.x = v[rr][c * V]; q.y = v[rr][c * V + 1]; }
            *reinterpret_cast<VT*>(sp + ((rr * (C / V) + c) * 32 + lane) * V) = q;
        }
}

// one row (the H values) in the first half of a state slot
template <typename T, int C>
__device__ __forceinline__ void strip_lds_half(const T* __restrict__ sp, int lane, T (&v)[C]) {
    constexpr int V = VecOf<T>::V;
    using VT = typename VecOf<T>::type;
#pragma unroll
    for (int c = 0; c < C / V; ++c) {
        const VT q = *reinterpret_cast<const VT*>(sp + (c * 32 + lane) * V);
        if constexpr (V == 4) { v[c * V] = q.x; v[c * V + 1] = q.y; v[c * V + 2] = q.z; v[c * V + 3] = q.w; }
        else { v[c * V] = q.x; v[c * V + 1] = q.y; }
    }
}
template <typename T, int C>
__device__ __forceinline__ void strip_sts_half(T* __restrict__ sp, int lane, const T (&v)[C]) {
    constexpr int V = VecOf<T>::V;
    using VT = typename VecOf<T>::type;
#pragma unroll
    for (int c = 0; c < C / V; ++c) {
        VT q;
        if constexpr (V == 4) { q.x = v[c * V]; q.y = v[c * V + 1]; q.z = v[c * V + 2]; q.w = v[c * V + 3]; }
        else { q.x = v[c * V]; q.y = v[c * V + 1]; }
        *reinterpret_cast<VT*>(sp + (c * 32 + lane) * V) = q;
    }
}

// Row pairs travel HBM -> shared memory with cp.async (16 bytes per lane into the lane-private slots; a
// slot is read by its owner lane after cp.async.wait_group and a __syncwarp, since with C/V > 1 another
// lane of the warp may have issued the copy) through a
// ring of kStripRing pairs: a pair is requested kStripRing-1 iterations before it is used, no register
// holds data in flight, and nothing has to be moved while a load is pending.
constexpr int kStripRing = GE_STRIP_RING;

__device__ __forceinline__ void cp_async16(void* smem_dst, const void* gmem_src) {
    asm volatile("cp.async.cg.shared.global [%0], [%1], 16;" ::"r"((uint32_t)__cvta_generic_to_shared(smem_dst)),
                 "l"(gmem_src) : "memory");
}
__device__ __forceinline__ void cp_async_commit() { asm volatile("cp.async.commit_group;" ::: "memory"); }
template <int N>
__device__ __forceinline__ void cp_async_wait() { asm volatile("cp.async.wait_group %0;" ::"n"(N) : "memory"); }

// request rows y, y+1 of the lane's columns into the pair slot `dst` (layout of strip_sts)
template <typename T, int C>
__device__ __forceinline__ void strip_request_pair(const T* __restrict__ uin, int nx, int ny, T ylo, T yhi, int y,
                                                   int e0, T* __restrict__ dst, int lane) {
    constexpr int V = VecOf<T>::V;
    using VT = typename VecOf<T>::type;
#pragma unroll
    for (int rr = 0; rr < 2; ++rr) {
        const int yy = y + rr;
        if ((unsigned)yy < (unsigned)ny) {
            // the warp copies the row's 32*C values as C/V instructions of 32 CONSECUTIVE 16-byte chunks
            // (full sectors on the global side); chunk q belongs to lane q / (C/V), vector q % (C/V)
            const T* __restrict__ row = uin + (int64_t)yy * nx + (e0 - lane * C);
#pragma unroll
            for (int cc = 0; cc < C / V; ++cc) {
                const int q = cc * 32 + lane;
                cp_async16(dst + ((rr * (C / V) + q % (C / V)) * 32 + q / (C / V)) * V, row + q * V);
            }
        } else {
            const T f = yy == -1 ? ylo : (yy == ny ? yhi : T(0));
            VT q;
            if constexpr (V == 4) { q.x = f; q.y = f; q.z = f; q.w = f; } else { q.x = f; q.y = f; }
#pragma unroll
            for (int c = 0; c < C / V; ++c) *reinterpret_cast<VT*>(dst + ((rr * (C / V) + c) * 32 + lane) * V) = q;
        }
    }
}

// The TB stages of one iteration: `cur` (raw pair of level 0, rows y0, y0+1; cx its column 0) flows through
// and comes out as the level-TB pair.  PURE: every group row (j = y0-1-l) is interior now and at the next
// iteration, so there is neither an edge test nor a raw slot; otherwise each stage decides (warp-uniform).
template <typename T, int C, int TB, bool BC, bool PURE, int COOP = 1>
__device__ __forceinline__ void strip_stages(T (&cur)[2][C], T (&cx)[2], T (&px)[TB][2], T* __restrict__ sp, int lane,
                                             const Strip2dCtx<T>& k, const Coef2<T>* __restrict__ coef, int y0, int ny,
                                             int par = 0) {
    constexpr int kPair = 2 * 32 * C;
#pragma unroll
    for (int l = 0; l < TB; ++l) {
        const int j = y0 - 1 - l;                                                  // group rows j, j+1
        const bool fast = PURE || (unsigned)j < (unsigned)(ny - 1);                // both interior
        const bool next_fast = PURE || (unsigned)(j + 2) < (unsigned)(ny - 1);     // this stage, next iteration
        T* slot = sp + l * kPair;
        T N[2][C], nx0[2] = {T(0), T(0)};
        T Hn[C], Rc[C / 2], Rd[C / 2];
        strip_rhs_pair<T, C>(cur[0], cur[1], k.r, Hn, Rc, Rd);
        if (fast) {
            T H[C];
            strip_lds_half<T, C>(slot, lane, H);
            if ((l & 1) != 0) strip_stage_L<T, C, BC, COOP>(H, Rc, Rd, px[l], cx, N[0], N[1], k, par);
            else              strip_stage_R<T, C, BC, COOP>(H, Rc, Rd, N[0], N[1], nx0, k, par);
        } else {
            T P[2][C];
            strip_lds<T, C>(slot, lane, P);
            strip_stage_rows<T, C, BC, COOP>((l & 1) != 0, P, px[l], cur, cx, N, nx0, k, coef, j, ny);
        }
        if (next_fast) strip_sts_half<T, C>(slot, lane, Hn);
        else           strip_sts<T, C>(slot, lane, cur);
#pragma unroll
        for (int s = 0; s < C; ++s) { cur[0][s] = N[0][s]; cur[1][s] = N[1][s]; }
        if constexpr (BC) { px[l][0] = cx[0]; px[l][1] = cx[1]; cx[0] = nx0[0]; cx[1] = nx0[1]; }
    }
}

template <typename T, int C, int TB, bool BC, int COOP = 1>
__device__ __forceinline__ void strip_run(const T* __restrict__ uin, T* __restrict__ uout, int nx, int ny,
                                          const Coef2<T>* __restrict__ coef, T* __restrict__ sp, int a0,
                                          int out_lo, int out_hi, bool first, bool last, int ys, int ye,
                                          int lane, int warp = 0, T* __restrict__ xch = nullptr) {
    constexpr int V = VecOf<T>::V;
    constexpr int kPair = 2 * 32 * C;             // elements of one row pair of the strip
    static_assert(TB % 2 == 0 && C % 2 == 0 && C % V == 0, "TB even; C holds whole groups and vectors");
    const Coef2<T> kk = *coef;
    Strip2dCtx<T> k;
    k.r = kk.r; k.g2 = kk.g2; k.g4 = kk.g4; k.h1 = kk.h1; k.h3 = kk.h3; k.xlo = kk.xlo; k.xhi = kk.xhi;
    k.warp = warp; k.gl = warp * 32 + lane; k.xch = xch; k.xslow = xch + StripXch<COOP>::lines;
    k.is_lo = BC && first && k.gl == 0; k.is_hi = BC && last && k.gl == COOP * 32 - 1;
    const int e0 = a0 + k.gl * C;
    const int Y0 = ys - TB;                       // first row pair that enters the pipeline
    constexpr int kLag = TB;                      // rows between the pair that enters and the pair that leaves
    const int iters = (ye - ys + 1) / 2 + TB;

    {
        T z[2][C];
#pragma unroll
        for (int j = 0; j < C; ++j) { z[0][j] = T(0); z[1][j] = T(0); }
#pragma unroll
        for (int l = 0; l < TB; ++l) strip_sts<T, C>(sp + l * kPair, lane, z);
    }
    T px[TB][2];                                  // column 0 of the previous pairs (lane is_lo, odd levels)
#pragma unroll
    for (int l = 0; l < TB; ++l) { px[l][0] = T(0); px[l][1] = T(0); }
    T* ring = sp + TB * kPair;                    // kStripRing pair slots after the TB state slots
#pragma unroll
    for (int q = 0; q < kStripRing - 1; ++q) {
        strip_request_pair<T, C>(uin, nx, ny, kk.ylo, kk.yhi, Y0 + 2 * q, e0, ring + q * kPair, lane);
        cp_async_commit();
    }

    // loop-carried bookkeeping instead of per-iteration multiplies and modulos: ring slots of the pair to
    // request / to read, element offsets of the rows to request / to write (64-bit, may run outside the grid:
    // only used under the row tests)
    int rq = kStripRing - 1, rd = 0;
    int64_t in_off = (int64_t)(Y0 + 2 * (kStripRing - 1)) * nx + e0;
    int64_t out_off = (int64_t)(Y0 - kLag) * nx + e0;
    bool st_ok[C / V];
#pragma unroll
    for (int c = 0; c < C / V; ++c) st_ok[c] = e0 + c * V >= out_lo && e0 + c * V < out_hi;
#pragma unroll 1
    for (int it = 0; it < iters; ++it, in_off += 2 * (int64_t)nx, out_off += 2 * (int64_t)nx) {
        const int y0 = Y0 + 2 * it;
        // request the pair of iteration it + kStripRing - 1 (its slot was read in iteration it - 1)
        if constexpr (C / V > 1) __syncwarp();    // by its owner lanes, which may not be the lanes that refill it
        {
            const int yq = y0 + 2 * (kStripRing - 1);
            T* dst = ring + rq * kPair;
            if (C == V && yq >= 0 && yq + 1 < ny) {        // both rows inside the grid (warp-uniform)
                cp_async16(dst + lane * V, uin + in_off);
                cp_async16(dst + (32 + lane) * V, uin + in_off + nx);
            } else {
                strip_request_pair<T, C>(uin, nx, ny, kk.ylo, kk.yhi, yq, e0, dst, lane);
            }
            rq = rq + 1 == kStripRing ? 0 : rq + 1;
        }
        cp_async_commit();
        cp_async_wait<kStripRing - 1>();          // the pair of this iteration has landed (this lane's copies)
        if constexpr (C / V > 1) __syncwarp();    // ... and the other lanes' copies into this lane's slots
        T cur[2][C], cx[2] = {T(0), T(0)};
        strip_lds<T, C>(ring + rd * kPair, lane, cur);
        rd = rd + 1 == kStripRing ? 0 : rd + 1;
        // every stage's group row interior now and at its next iteration: the pure pipeline, no edge tests
        if (y0 - TB >= 0 && y0 + 1 < ny - 1) strip_stages<T, C, TB, BC, true, COOP>(cur, cx, px, sp, lane, k, coef, y0, ny, it & 1);
        else                                 strip_stages<T, C, TB, BC, false, COOP>(cur, cx, px, sp, lane, k, coef, y0, ny, it & 1);
        // cur holds level-TB rows (y0 - kLag, y0 - kLag + 1), unshifted (TB is even)
        if (it >= kLag) {
            const int yo = y0 - kLag;
#pragma unroll
            for (int rr = 0; rr < 2; ++rr) {
                if (yo + rr < ye) {
                    T* __restrict__ row = uout + out_off + (rr ? nx : 0);
#pragma unroll
                    for (int c = 0; c < C / V; ++c) {
                        if (st_ok[c]) {
                            T t[V];
#pragma unroll
                            for (int q = 0; q < V; ++q) t[q] = cur[rr][c * V + q];
                            st_vec(row + c * V, t);
                        }
                    }
                }
            }
        }
    }
}

// resident CTAs per SM the register allocation is held to (measured r01: tighter caps spill and lose
// 3x; -DGE_STRIP_MINB_F32/F64 through GE_NVCC_EXTRA for sweeps)
#ifndef GE_STRIP_MINB_F32
#define GE_STRIP_MINB_F32 3
#endif
#ifndef GE_STRIP_MINB_F64
#define GE_STRIP_MINB_F64 4
#endif
template <typename T> struct StripMinBlocks { static constexpr int n = sizeof(T) == 8 ? GE_STRIP_MINB_F64 : GE_STRIP_MINB_F32; };

template <typename T, int C, int TB>
__global__ void __launch_bounds__(kStripWarps * 32, StripMinBlocks<T>::n)
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
    extern __shared__ __align__(16) unsigned char strip_smem[];
    T* sp = reinterpret_cast<T*>(strip_smem) + (size_t)warp * (TB + kStripRing) * 2 * 32 * C;   // state + ring of this warp
    if (first || last) strip_run<T, C, TB, true>(uin, uout, nx, ny, coef, sp, a0, out_lo, out_hi, first, last, ys, ye, lane);
    else               strip_run<T, C, TB, false>(uin, uout, nx, ny, coef, sp, a0, out_lo, out_hi, false, false, ys, ye, lane);
}

// Host launcher: TB levels starting at a PHASE-1 level; `configured` is the caller's per-plan flag for
// this instantiation's function attributes.  Requires nx % V == 0, nx even, nx >= 32*C,
// 16-byte aligned buffers and nx, ny < 2^30.
template <typename T, int C, int TB>
inline cudaError_t strip2d_launch(const T* uin, T* uout, int64_t nx, int64_t ny, const Coef2<T>* coef, int hp,
                                  bool& configured, cudaStream_t s) {
    const Strip2dGeom g = strip2d_geom(C, VecOf<T>::V, TB, nx, ny, hp);
    dim3 grid((unsigned)((g.nstrips + kStripWarps - 1) / kStripWarps), (unsigned)g.segs);
    constexpr size_t smem = (size_t)kStripWarps * (TB + kStripRing) * 2 * 32 * C * sizeof(T);
    // once per plan (= per device) and instantiation: allow > 48 KB and the full carve-out
    if (!configured) {
        cudaError_t e = cudaFuncSetAttribute(ge2d_strip_kernel<T, C, TB>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
        if (e == cudaSuccess) e = cudaFuncSetAttribute(ge2d_strip_kernel<T, C, TB>, cudaFuncAttributePreferredSharedMemoryCarveout, 100);
        if (e != cudaSuccess) return e;
        configured = true;
    }
    ge2d_strip_kernel<T, C, TB><<<grid, kStripWarps * 32, smem, s>>>(uin, uout, (int)nx, (int)ny, coef, g);
    return cudaGetLastError();
}

// ---- cooperative form: the CTA's COOP warps own ONE strip of COOP*32*C columns (strip_neighbour) ----
inline Strip2dGeom strip2d_coop_geom(int C, int V, int TB, int COOP, int64_t nx, int64_t ny, int hp) {
    Strip2dGeom g;
    const int64_t w = (int64_t)COOP * 32 * C;
    g.halo = (TB + V - 1) / V * V;
    g.valid = (int)(w - 2 * g.halo);
    g.nreg = 1 + (int)((nx + g.halo - w) / g.valid);
    g.nstrips = g.nreg + 1;
    g.hp = hp;
    g.segs = (int)((ny + 2 * (int64_t)hp - 1) / (2 * (int64_t)hp));
    return g;
}

template <typename T, int C, int TB, int COOP>
__global__ void __launch_bounds__(COOP * 32, 16 / COOP)     // 16 resident warps per SM, as for the plain kernel
ge2d_strip_coop_kernel(const T* __restrict__ uin, T* __restrict__ uout, int nx, int ny,
                       const Coef2<T>* __restrict__ coef, const Strip2dGeom g) {
    const int lane = threadIdx.x & 31;
    const int warp = threadIdx.x >> 5;
    const int strip = blockIdx.x;
    const bool first = strip == 0, last = strip == g.nreg;
    const int a0 = first ? 0 : (last ? nx - COOP * 32 * C : strip * g.valid - g.halo);
    const int out_lo = strip * g.valid;
    const int out_hi = last ? nx : out_lo + g.valid;
    const int ys = 2 * g.hp * (int)blockIdx.y;
    const int ye = ys + 2 * g.hp < ny ? ys + 2 * g.hp : ny;
    extern __shared__ __align__(16) unsigned char strip_smem[];
    T* xch = reinterpret_cast<T*>(strip_smem);
    T* sp = xch + StripXch<COOP>::elems + (size_t)warp * (TB + kStripRing) * 2 * 32 * C;   // state + ring of this warp
    if (first || last) strip_run<T, C, TB, true, COOP>(uin, uout, nx, ny, coef, sp, a0, out_lo, out_hi, first, last, ys, ye, lane, warp, xch);
    else               strip_run<T, C, TB, false, COOP>(uin, uout, nx, ny, coef, sp, a0, out_lo, out_hi, false, false, ys, ye, lane, warp, xch);
}

// Host launcher of the cooperative form; requires nx >= COOP*32*C on top of strip2d_launch's conditions.
template <typename T, int C, int TB, int COOP>
inline cudaError_t strip2d_coop_launch(const T* uin, T* uout, int64_t nx, int64_t ny, const Coef2<T>* coef, int hp,
                                       bool& configured, cudaStream_t s) {
    const Strip2dGeom g = strip2d_coop_geom(C, VecOf<T>::V, TB, COOP, nx, ny, hp);
    dim3 grid((unsigned)g.nstrips, (unsigned)g.segs);
    constexpr size_t smem = ((size_t)COOP * (TB + kStripRing) * 2 * 32 * C + StripXch<COOP>::elems) * sizeof(T);
    if (!configured) {
        cudaError_t e = cudaFuncSetAttribute(ge2d_strip_coop_kernel<T, C, TB, COOP>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
        if (e == cudaSuccess) e = cudaFuncSetAttribute(ge2d_strip_coop_kernel<T, C, TB, COOP>, cudaFuncAttributePreferredSharedMemoryCarveout, 100);
        if (e != cudaSuccess) return e;
        configured = true;
    }
    ge2d_strip_coop_kernel<T, C, TB, COOP><<<grid, COOP * 32, smem, s>>>(uin, uout, (int)nx, (int)ny, coef, g);
    return cudaGetLastError();
}

}  // namespace ge
