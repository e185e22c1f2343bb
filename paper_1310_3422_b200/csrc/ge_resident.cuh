// ge_resident.cuh -- strategy C (1-D): the state stays in REGISTERS for the
// whole run; HBM is touched once at the start and once at the end.
//
// This is the Blackwell answer to the paper's synchronisation question
// (one thread per sub-domain couple, two block barriers per
// level pair, and no correct barrier ACROSS blocks -- PAPER.md:160, :216).
// Two kernels share one level code:
//
//   (i)  ge1d_rod_resident_kernel   a rod (nx <= 32*C*W nodes) lives in one CTA
//        of W warps, C values per lane.  W = 1: no barrier at all, one warp
//        shuffle per lane and level.  W > 1: the two warp-edge values cross
//        through shared memory, one __syncthreads per level.  Batched rods
//        (SURVEY.md 8(a) a6): one rod per CTA, loaded once, marched `steps`
//        levels, stored once.
//   (ii) ge1d_grid_resident_kernel  ONE long rod spread over the whole chip by a
//        cooperative launch: a warp owns a tile of (32-2*hl)*C nodes plus hl
//        halo lanes on either side.  The halo goes stale by one node per level
//        (below), so tiles only meet every tb <= hl*C levels: each warp
//        publishes its outermost valid lanes to a small L2-resident exchange
//        buffer and refreshes its halo lanes from its two neighbours'.  The
//        meeting is either NEIGHBOUR-ONLY (a release/acquire flag per tile --
//        the paper's observation that only wall nodes are shared,
//        PAPER.md:138) or a GRID-WIDE barrier (cooperative groups), selectable
//        for the comparison north_star asks for.
//
// Level code (drift-free sliding window).  In the "even state" lane t holds
// the window [w, w+C), w even.  Levels come in pairs:
//   R  (phase 1: left members at odd elements)  the lane updates the pairs
//      (w+1,w+2) ... (w+C-1,w+C); the last pair's right-hand side q comes from
//      the next lane (one shuffle); the window becomes [w+1, w+C+1).
//   L  (phase 0: left members at even elements, i.e. again at odd SLOTS of the
//      shifted window)  the lane updates (w,w+1) ... (w+C-2,w+C-1); the first
//      pair's left right-hand side p comes from the previous lane (one
//      shuffle); the window is [w, w+C) again.
// So a pair of levels costs two shuffles and no register moves, and the
// arithmetic is the 3-flop-per-node factored form of ge_temporal.cuh (the
// difference e across a group boundary is shared by the two adjacent pairs) --
// the same expression tree as every other libge kernel, so results are
// bit-identical to the per-level kernel.
// A run that starts at a phase-0 level first takes one in-lane level I (pairs
// (w,w+1) ..., two shuffles); a run with one level left over takes R followed
// by a one-slot shift back.
//
// Validity.  A window edge that lies ON a group boundary loses one node per
// level: the pair that straddles it in the next (shifted) pattern cannot be
// formed.  After n levels a lane group that started fully valid has n stale
// nodes on either side (I and the shift back are counted as 2).
//
// Boundaries.  nx % C == 0 is required, so element 0 is
// slot 0 of some lane (`is_lo`) and element nx-1 is slot C-1 of some lane
// (`is_hi`); the Dirichlet values never occupy a slot of a valid lane:
//   R: node 1 is single: new = z0 - e (z0 - beta_lo) (Eq (1));
//      it leaves the shifted window and is kept in the extra register x0.
//      The last pair of lane is_hi is (N, N+1): q := beta_hi, g := e (Eq (2)).
//   L: the first pair of lane is_lo is (1,2): its p is formed from x0 and
//      beta_lo instead of the shuffled value.
// Lanes outside the rod hold finite filler and never feed a valid lane.
#pragma once
#include <cooperative_groups.h>

#include "ge_common.cuh"

namespace ge {

namespace cg = cooperative_groups;

template <typename T>
__device__ __forceinline__ void ld_vec_plain(const T* p, T (&x)[VecOf<T>::V]) {
    using VT = typename VecOf<T>::type;
    const VT v = *reinterpret_cast<const VT*>(p);
    if constexpr (VecOf<T>::V == 4) { x[0] = v.x; x[1] = v.y; x[2] = v.z; x[3] = v.w; }
    else { x[0] = v.x; x[1] = v.y; }
}
template <typename T>
__device__ __forceinline__ void ld_vec_cg(const T* p, T (&x)[VecOf<T>::V]) {
    using VT = typename VecOf<T>::type;
    const VT v = __ldcg(reinterpret_cast<const VT*>(p));
    if constexpr (VecOf<T>::V == 4) { x[0] = v.x; x[1] = v.y; x[2] = v.z; x[3] = v.w; }
    else { x[0] = v.x; x[1] = v.y; }
}
template <typename T>
__device__ __forceinline__ void st_vec_cg(T* p, const T (&x)[VecOf<T>::V]) {
    using VT = typename VecOf<T>::type;
    VT v;
    if constexpr (VecOf<T>::V == 4) { v.x = x[0]; v.y = x[1]; v.z = x[2]; v.w = x[3]; }
    else { v.x = x[0]; v.y = x[1]; }
    __stcg(reinterpret_cast<VT*>(p), v);
}

// Per-lane constants of the resident level code.  XW: the W > 1 warps of the CTA hold one rod and
// exchange their edge values through shared memory (sx: [2 buffers][2 sides][nwarps]).
template <typename T, bool XW>
struct ResidentCtx {
    T r, g, e, lo, hi;
    bool is_lo, is_hi;
    int lane, warp, nwarps;
    T* sx;
};

// value `mine` of lane+1 (next warp's lane 0 through shared memory when XW)
template <typename T, bool XW>
__device__ __forceinline__ T from_right(const ResidentCtx<T, XW>& c, T mine, int buf) {
    T got = __shfl_down_sync(0xffffffffu, mine, 1);
    if constexpr (XW) {
        T* slot = c.sx + (buf * 2 + 0) * c.nwarps;
        if (c.lane == 0) slot[c.warp] = mine;
        __syncthreads();
        if (c.lane == 31 && c.warp + 1 < c.nwarps) got = slot[c.warp + 1];
    }
    return got;
}
// value `mine` of lane-1 (previous warp's lane 31 through shared memory when XW)
template <typename T, bool XW>
__device__ __forceinline__ T from_left(const ResidentCtx<T, XW>& c, T mine, int buf) {
    T got = __shfl_up_sync(0xffffffffu, mine, 1);
    if constexpr (XW) {
        T* slot = c.sx + (buf * 2 + 1) * c.nwarps;
        if (c.lane == 31) slot[c.warp] = mine;
        __syncthreads();
        if (c.lane == 0 && c.warp > 0) got = slot[c.warp - 1];
    }
    return got;
}

// R: even state -> shifted state, left members at odd slots (a phase-1 level).  In place.
// BC = false: the lane group holds no boundary (interior tiles of ge_temporal.cuh): the boundary
// selects and the x0 bookkeeping drop out at compile time.
template <typename T, int C, bool XW, bool BC = true>
__device__ __forceinline__ void level_R(T (&v)[C], T& x0, const ResidentCtx<T, XW>& c, int buf) {
    const T r = c.r, g = c.g;
    T e = v[1] - v[0];
    T pprev = fma(-r, e, v[1]);               // rhs of Eq (2) at the left member in slot 1
    const T z0 = fma(r, e, v[0]);             // rhs of Eq (1) at the right member in slot 0
    const T zin = from_right<T, XW>(c, z0, buf);
    // node 1 when it is single (partner is node 0): only lane is_lo reads x0 later
    if constexpr (BC) x0 = fma(-c.e, z0 - c.lo, z0);
#pragma unroll
    for (int m = 1; m < C / 2; ++m) {
        e = v[2 * m + 1] - v[2 * m];
        const T pm = fma(-r, e, v[2 * m + 1]);
        const T zm = fma(r, e, v[2 * m]);
        const T t = zm - pprev;               // pair (slots 2m-1, 2m): q = z_m, p = p_{m-1}
        v[2 * m - 2] = fma(g, t, pprev);
        v[2 * m - 1] = fma(-g, t, zm);
        pprev = pm;
    }
    const bool hi = BC && c.is_hi;
    const T ql = hi ? c.hi : zin;             // (N, N+1): the boundary value is the new-level neighbour
    const T gl = hi ? c.e : g;
    const T t = ql - pprev;
    v[C - 2] = fma(gl, t, pprev);
    const T last = fma(-gl, t, ql);
    v[C - 1] = hi ? c.hi : last;              // the ghost stays pinned
}

// L: shifted state -> even state, left members at odd slots of the shifted window (a phase-0 level).
template <typename T, int C, bool XW, bool BC = true>
__device__ __forceinline__ void level_L(T (&v)[C], const T x0, const ResidentCtx<T, XW>& c, int buf) {
    const T r = c.r, g = c.g;
    T e = v[C - 1] - v[C - 2];
    const T plast = fma(-r, e, v[C - 1]);     // p of the pair this lane hands to the next one
    T znext = fma(r, e, v[C - 2]);
    const T pin = from_left<T, XW>(c, plast, buf);
#pragma unroll
    for (int m = C / 2 - 2; m >= 0; --m) {
        e = v[2 * m + 1] - v[2 * m];
        const T pm = fma(-r, e, v[2 * m + 1]);
        const T zm = fma(r, e, v[2 * m]);
        const T t = znext - pm;               // pair (slots 2m+1, 2m+2) lands in slots 2m+2, 2m+3
        v[2 * m + 2] = fma(g, t, pm);
        v[2 * m + 3] = fma(-g, t, znext);
        znext = zm;
    }
    T P = pin;
    if constexpr (BC) {
        const T pl = fma(-r, x0 - c.lo, x0);  // pair (1,2): left member is x0, its left neighbour node 0
        P = c.is_lo ? pl : pin;
    }
    const T t = znext - P;
    v[0] = fma(g, t, P);
    v[1] = fma(-g, t, znext);
}

// I: even state -> even state, pairs (slots 2m, 2m+1) inside the lane (a phase-0 level).
template <typename T, int C, bool XW, bool BC = true>
__device__ __forceinline__ void level_I(T (&v)[C], const ResidentCtx<T, XW>& c, int buf) {
    const T r = c.r, g = c.g;
    T a = from_left<T, XW>(c, v[C - 1], buf);
    T d = from_right<T, XW>(c, v[0], buf);
    if (BC && c.is_lo) a = c.lo;
    if (BC && c.is_hi) d = c.hi;
#pragma unroll
    for (int m = 0; m < C / 2; ++m) {
        const T b = v[2 * m], cc = v[2 * m + 1];
        const T dd = (m == C / 2 - 1) ? d : v[2 * m + 2];
        const T p = fma(r, a - b, b);
        const T q = fma(r, dd - cc, cc);
        const T t = q - p;
        a = cc;
        v[2 * m] = fma(g, t, p);
        v[2 * m + 1] = fma(-g, t, q);
    }
}

// shifted state -> even state without a level (after a lone R at the end of a run)
template <typename T, int C, bool XW, bool BC = true>
__device__ __forceinline__ void unshift(T (&v)[C], const T x0, const ResidentCtx<T, XW>& c, int buf) {
    T left = from_left<T, XW>(c, v[C - 1], buf);
    if (BC && c.is_lo) left = x0;
#pragma unroll
    for (int j = C - 1; j >= 1; --j) v[j] = v[j - 1];
    v[0] = left;
}

// ------------------------------------------------------------------ (i) rod per CTA ------
template <typename T, int C, int W>
__global__ void __launch_bounds__(32 * W)
ge1d_rod_resident_kernel(T* u, int64_t nx, int64_t batch, const Coef1<T>* __restrict__ coef,
                         int phase0, int64_t steps) {
    constexpr int V = VecOf<T>::V;
    constexpr bool XW = W > 1;
    static_assert(C % 2 == 0 && C % V == 0, "C must hold whole pairs and whole vectors");
    __shared__ T sx[4 * W];
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    const int gl = warp * 32 + lane;                 // lane index within the rod
    const int used = (int)(nx / C);                  // lanes that hold nodes
    for (int64_t rod = blockIdx.x; rod < batch; rod += gridDim.x) {
        const Coef1<T> k = coef[rod];
        ResidentCtx<T, XW> c;
        c.r = k.r; c.g = k.g; c.e = k.e; c.lo = k.lo; c.hi = k.hi;
        c.is_lo = gl == 0; c.is_hi = gl == used - 1;
        c.lane = lane; c.warp = warp; c.nwarps = W; c.sx = sx;
        T* row = u + rod * nx + (int64_t)gl * C;
        T v[C];
        T x0 = T(0);
        if (gl < used) {
#pragma unroll
            for (int j = 0; j < C / V; ++j) {
                T t[V];
                ld_vec_plain(row + j * V, t);
#pragma unroll
                for (int i = 0; i < V; ++i) v[j * V + i] = t[i];
            }
        } else {
#pragma unroll
            for (int j = 0; j < C; ++j) v[j] = k.hi;
        }
        int64_t left = steps;
        int buf = 0;
        if (phase0 == 0 && left > 0) { level_I<T, C, XW>(v, c, buf); buf ^= 1; --left; }
#pragma unroll 1
        for (; left >= 2; left -= 2) {
            level_R<T, C, XW>(v, x0, c, buf);
            level_L<T, C, XW>(v, x0, c, buf ^ 1);
        }
        if (left) {
            level_R<T, C, XW>(v, x0, c, buf);
            unshift<T, C, XW>(v, x0, c, buf ^ 1);
        }
        if (gl < used) {
#pragma unroll
            for (int j = 0; j < C / V; ++j) {
                T t[V];
#pragma unroll
                for (int i = 0; i < V; ++i) t[i] = v[j * V + i];
                st_vec(row + j * V, t);
            }
        }
        if constexpr (XW) __syncthreads();           // the exchange slots are reused by the next rod
    }
}

template <typename T, int C, int W>
inline cudaError_t rod_resident_launch(T* u, int64_t nx, int64_t batch, const Coef1<T>* coef, int phase0,
                                       int64_t steps, cudaStream_t s) {
    const unsigned grid = (unsigned)(batch < (1 << 30) ? batch : (1 << 30));
    ge1d_rod_resident_kernel<T, C, W><<<grid, 32 * W, 0, s>>>(u, nx, batch, coef, phase0, steps);
    return cudaGetLastError();
}

// ------------------------------------------------------------------ (ii) one rod on the whole chip ------
constexpr int kGridWarps = 4;              // warps (tiles) per CTA
// how the tiles meet: 0 = per-tile flag with a release fence (neighbours only), 1 = grid-wide barrier,
// 2 = flag-in-data lines, no fence and no separate flag (neighbours only), 3 = the same, published every
// tb/2 levels and consumed in opposite turns by the CTAs that share an SM
constexpr int kSyncFlags = 0, kSyncGrid = 1, kSyncLL = 2, kSyncStagger = 3;
// 4 .. 7 = thread-block CLUSTERS of 2 / 4 / 8 / 16 CTAs (kernel instantiation CL = true): the tiles of a cluster
// publish into their CTA's shared memory, meet at the cluster's hardware barrier and read their neighbours' sides
// from shared memory -- their own CTA's or, through distributed shared memory, the adjacent CTA's; only the two
// tiles at the ends of a cluster exchange through L2, with flag-in-data lines as in mode 2
constexpr int kSyncCluster2 = 4, kSyncCluster16 = 7;
inline int sync_cluster_size(int mode) { return mode >= kSyncCluster2 && mode <= kSyncCluster16 ? 2 << (mode - kSyncCluster2) : 1; }
constexpr int kLineSlots = 4;          // exchange slots of the flag-in-data modes (2 are used by kSyncLL)

struct GridResidentArgs {
    int64_t nx;
    int64_t ntiles;
    int64_t steps;
    int phase0;
    int hl;            // halo lanes per side
    int tb;            // levels between two meetings, <= hl*C
    int sync_mode;     // kSyncFlags / kSyncGrid / kSyncLL
    unsigned epoch0;   // flag value all tiles had when the launch started
};

// number of meetings of a run (the same loop as in the kernel); host and device
__host__ __device__ inline int64_t grid_resident_meetings(int64_t steps, int phase0, int tb) {
    int64_t left = steps, n = 0;
    int usedl = 0;
    if (phase0 == 0 && left > 0) { usedl = 2; --left; }
    while (left >= 2) {
        if (usedl + 2 > tb) { ++n; usedl = 0; }
        usedl += 2; left -= 2;
    }
    if (left) { if (usedl + 2 > tb) { ++n; usedl = 0; } }
    return n;
}

// publications of a staggered run (the same loop as in the kernel) + the final one
__host__ __device__ inline int64_t grid_resident_halves(int64_t steps, int phase0, int tb) {
    const int tbh = tb / 2 - (tb / 2) % 2;
    int64_t left = steps, n = 0;
    int usedh = 0;
    if (phase0 == 0 && left > 0) { usedh = 2; --left; }
    while (left >= 2) {
        if (usedh + 2 > tbh) { ++n; usedh = 0; }
        usedh += 2; left -= 2;
    }
    if (left) { if (usedh + 2 > tbh) { ++n; usedh = 0; } }
    return n + 1;
}

__device__ __forceinline__ unsigned ld_acquire_u32(const unsigned* p) {
    unsigned v;      // LDG.STRONG.GPU + CCTL.IVALL: no MEMBAR on the reader's side
    asm volatile("ld.acquire.gpu.global.u32 %0, [%1];" : "=r"(v) : "l"(p) : "memory");
    return v;
}
__device__ __forceinline__ void st_relaxed_u32(unsigned* p, unsigned v) {
    asm volatile("st.relaxed.gpu.global.u32 [%0], %1;" ::"l"(p), "r"(v) : "memory");
}
// One lane spins until BOTH neighbours' flags have reached `target` (wrap-safe); the two loads of a
// round are in flight together.  Bounded: a tile that never arrives (which a cooperative launch rules
// out) ends the wait after ~1 s and is reported through `fault`.
__device__ __forceinline__ void wait_flags(const unsigned* pl, const unsigned* pr, unsigned target,
                                           unsigned* fault) {
    for (unsigned it = 0; it < (1u << 24); ++it) {
        const unsigned a = pl ? ld_acquire_u32(pl) : target;
        const unsigned b = pr ? ld_acquire_u32(pr) : target;
        if ((int)(a - target) >= 0 && (int)(b - target) >= 0) return;
        if (it > 4096) __nanosleep(64);
    }
    atomicExch(fault, 1u);
}

// Flag-in-data exchange lines (the scheme of low-latency collectives): every 8-byte unit carries 32
// bits of payload and the 32-bit meeting number, so a reader that sees the expected number in both
// units of a 16-byte line has the payload -- no fence, no separate flag, one L2 round trip.
// An fp64 value fills one line (lo, tag, hi, tag); two fp32 values share one.
__device__ __forceinline__ void st_line(uint4* p, unsigned a, unsigned b, unsigned tag) {
    asm volatile("st.relaxed.gpu.global.v4.u32 [%0], {%1,%2,%3,%4};" ::"l"(p), "r"(a), "r"(tag), "r"(b), "r"(tag)
                 : "memory");
}
__device__ __forceinline__ uint4 ld_line(const uint4* p) {
    uint4 q;
    asm volatile("ld.relaxed.gpu.global.v4.u32 {%0,%1,%2,%3}, [%4];"
                 : "=r"(q.x), "=r"(q.y), "=r"(q.z), "=r"(q.w) : "l"(p) : "memory");
    return q;
}
template <typename T> struct Line;
template <> struct Line<double> {
    static constexpr int per = 1;     // values per line
    static __device__ __forceinline__ void put(uint4* p, const double* x, unsigned tag) {
        st_line(p, (unsigned)__double2loint(x[0]), (unsigned)__double2hiint(x[0]), tag);
    }
    static __device__ __forceinline__ void get(const uint4 q, double* x) {
        x[0] = __hiloint2double((int)q.z, (int)q.x);
    }
};
template <> struct Line<float> {
    static constexpr int per = 2;
    static __device__ __forceinline__ void put(uint4* p, const float* x, unsigned tag) {
        st_line(p, __float_as_uint(x[0]), __float_as_uint(x[1]), tag);
    }
    static __device__ __forceinline__ void get(const uint4 q, float* x) {
        x[0] = __uint_as_float(q.x); x[1] = __uint_as_float(q.z);
    }
};

template <typename T, int C, bool CL = false>
__global__ void __launch_bounds__(32 * kGridWarps)
ge1d_grid_resident_kernel(T* u, T* xbuf, const Coef1<T>* __restrict__ coef, unsigned* flags, unsigned* fault,
                          const GridResidentArgs a) {
    constexpr int V = VecOf<T>::V;
    static_assert(C % 2 == 0 && C % V == 0, "C must hold whole pairs and whole vectors");
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    const int64_t tile = (int64_t)blockIdx.x * kGridWarps + warp;
    const bool active = tile < a.ntiles;
    const int hl = a.hl;
    const int64_t valid = (int64_t)(32 - 2 * hl) * C;
    const int64_t e0 = tile * valid + (int64_t)(lane - hl) * C;      // element in slot 0 (even state)
    const bool inside = active && e0 >= 0 && e0 < a.nx;
    const Coef1<T> k = coef[0];
    ResidentCtx<T, false> c;
    c.r = k.r; c.g = k.g; c.e = k.e; c.lo = k.lo; c.hi = k.hi;
    c.is_lo = active && e0 == 0; c.is_hi = active && e0 + C == a.nx;
    c.lane = lane; c.warp = warp; c.nwarps = kGridWarps; c.sx = nullptr;
    cg::grid_group grid = cg::this_grid();

    T v[C];
    T x0 = T(0);
    if (inside) {
#pragma unroll
        for (int j = 0; j < C / V; ++j) {
            T t[V];
            ld_vec_plain(u + e0 + j * V, t);
#pragma unroll
            for (int i = 0; i < V; ++i) v[j * V + i] = t[i];
        }
    } else {
        const T f = e0 < 0 ? k.lo : k.hi;
#pragma unroll
        for (int j = 0; j < C; ++j) v[j] = f;
    }
    // stage 0: every tile has read its window; nobody may overwrite u before its neighbours did
    unsigned stage = a.epoch0 + 1;
    const bool own_l = lane >= hl && lane < 2 * hl;                   // outermost valid lanes
    const bool own_r = lane >= 32 - 2 * hl && lane < 32 - hl;
    const bool halo_l = lane < hl, halo_r = lane >= 32 - hl;
    const bool has_l = active && tile > 0, has_r = active && tile + 1 < a.ntiles;
    const size_t side = (size_t)hl * C;                               // elements per published side
    auto signal = [&]() {
        if (a.sync_mode == kSyncGrid) { grid.sync(); return; }
        if (a.sync_mode == kSyncLL || a.sync_mode == kSyncStagger || !active) return;
        // release: the warp's stores are ordered before lane 0's fence by __syncwarp, the fence is cumulative
        __syncwarp();
        if (lane == 0) { __threadfence(); st_relaxed_u32(flags + tile, stage); }
    };
    auto await = [&]() {
        if (!(a.sync_mode == kSyncFlags || CL) || !active) return;
        // lane 0 acquires for the warp; __syncwarp orders the other lanes' reads after it
        if (lane == 0 && (has_l || has_r))
            wait_flags(has_l ? flags + tile - 1 : nullptr, has_r ? flags + tile + 1 : nullptr, stage, fault);
        __syncwarp();
    };
    signal();

    int parity = 0;
    constexpr int NQ = C / Line<T>::per;                              // lines per lane
    // flag-in-data: publish tagged lines into slot `slot` (of kLineSlots); consume = poll the neighbours' lines
    // of that slot until every tag matches
    auto publish_lines = [&](int slot, unsigned tag) {
        if (!active || !(own_l || own_r)) return;
        uint4* xl = reinterpret_cast<uint4*>(xbuf);
        const size_t lside = (size_t)hl * NQ;
        uint4* dst = xl + ((size_t)slot * a.ntiles + tile) * 2 * lside +
                     (own_l ? (size_t)(lane - hl) * NQ : lside + (size_t)(lane - (32 - 2 * hl)) * NQ);
#pragma unroll
        for (int j = 0; j < NQ; ++j) Line<T>::put(dst + j, &v[j * Line<T>::per], tag);
    };
    auto consume_lines = [&](int slot, unsigned tag) {
        if (!active) return;
        const uint4* xl = reinterpret_cast<const uint4*>(xbuf);
        const size_t lside = (size_t)hl * NQ;
        const uint4* src = nullptr;
        if (halo_l && has_l)
            src = xl + ((size_t)slot * a.ntiles + tile - 1) * 2 * lside + lside + (size_t)lane * NQ;
        else if (halo_r && has_r)
            src = xl + ((size_t)slot * a.ntiles + tile + 1) * 2 * lside + (size_t)(lane - (32 - hl)) * NQ;
        if (src) {
            uint4 q[NQ];
            bool ok = false;
            // watch the line written last with a back-off (a spinning lane would take issue slots from
            // the warp that shares this scheduler and is still computing), then fetch all of them
            for (unsigned it = 0; it < (1u << 22); ++it) {
                const uint4 w = ld_line(src + NQ - 1);
                if (w.y == tag && w.w == tag) break;
                __nanosleep(it < 64 ? 20 : 200);
            }
            for (unsigned it = 0; it < (1u << 20) && !ok; ++it) {
#pragma unroll
                for (int j = 0; j < NQ; ++j) q[j] = ld_line(src + j);
                ok = true;
#pragma unroll
                for (int j = 0; j < NQ; ++j) ok = ok && q[j].y == tag && q[j].w == tag;
                if (!ok) __nanosleep(100);
            }
            if (!ok) atomicExch(fault, 1u);
#pragma unroll
            for (int j = 0; j < NQ; ++j) Line<T>::get(q[j], &v[j * Line<T>::per]);
        }
        __syncwarp();
    };
    auto meet_lines = [&]() {
        ++stage;
        publish_lines(parity, stage);
        consume_lines(parity, stage);
        parity ^= 1;
    };
    // cluster meeting (CL): shared memory [2 parities][kGridWarps tiles][2 sides][hl*C]; double-buffered, so the one
    // cluster barrier of a meeting also orders the reads of the meeting before the last against the next writes
    auto meet_cluster = [&]() {
        if constexpr (CL) {
            extern __shared__ __align__(16) unsigned char gr_smem[];
            T* xs = reinterpret_cast<T*>(gr_smem);
            cg::cluster_group cluster = cg::this_cluster();
            const unsigned crank = cluster.block_rank(), csize = cluster.num_blocks();
            const bool cross_l = has_l && warp == 0 && crank == 0;                        // the neighbour is in another cluster
            const bool cross_r = has_r && warp == kGridWarps - 1 && crank == csize - 1;
            ++stage;
            if (active && (own_l || own_r)) {
                T* dst = xs + ((size_t)(parity * kGridWarps + warp) * 2 + (own_l ? 0 : 1)) * side +
                         (size_t)(own_l ? lane - hl : lane - (32 - 2 * hl)) * C;
#pragma unroll
                for (int j = 0; j < C / V; ++j) {
                    T t[V];
#pragma unroll
                    for (int i = 0; i < V; ++i) t[i] = v[j * V + i];
                    st_vec(dst + j * V, t);
                }
                // the side that faces another cluster also goes to L2 as flag-in-data lines (mode 2's exchange: payload
                // and meeting number in one 8-byte unit, no fence, no separate flag)
                if ((own_l && cross_l) || (own_r && cross_r)) {
                    uint4* xl = reinterpret_cast<uint4*>(xbuf);
                    const size_t lside = (size_t)hl * NQ;
                    uint4* ldst = xl + ((size_t)parity * a.ntiles + tile) * 2 * lside +
                                  (own_l ? (size_t)(lane - hl) * NQ : lside + (size_t)(lane - (32 - 2 * hl)) * NQ);
#pragma unroll
                    for (int j = 0; j < NQ; ++j) Line<T>::put(ldst + j, &v[j * Line<T>::per], stage);
                }
            }
            cluster.sync();
            if (active) {
                const T* src = nullptr;
                const uint4* lsrc = nullptr;
                if (halo_l && has_l) {
                    if (cross_l) lsrc = reinterpret_cast<const uint4*>(xbuf) + ((size_t)parity * a.ntiles + tile - 1) * 2 * ((size_t)hl * NQ) +
                                        (size_t)hl * NQ + (size_t)lane * NQ;
                    else {
                        const T* base = warp > 0 ? xs : cluster.map_shared_rank(xs, crank - 1);
                        const int w = warp > 0 ? warp - 1 : kGridWarps - 1;
                        src = base + ((size_t)(parity * kGridWarps + w) * 2 + 1) * side + (size_t)lane * C;
                    }
                } else if (halo_r && has_r) {
                    if (cross_r) lsrc = reinterpret_cast<const uint4*>(xbuf) + ((size_t)parity * a.ntiles + tile + 1) * 2 * ((size_t)hl * NQ) +
                                        (size_t)(lane - (32 - hl)) * NQ;
                    else {
                        const T* base = warp < kGridWarps - 1 ? xs : cluster.map_shared_rank(xs, crank + 1);
                        const int w = warp < kGridWarps - 1 ? warp + 1 : 0;
                        src = base + ((size_t)(parity * kGridWarps + w) * 2 + 0) * side + (size_t)(lane - (32 - hl)) * C;
                    }
                }
                if (src) {
#pragma unroll
                    for (int j = 0; j < C / V; ++j) {
                        T t[V];
                        ld_vec_plain(src + j * V, t);
#pragma unroll
                        for (int i = 0; i < V; ++i) v[j * V + i] = t[i];
                    }
                }
                if (lsrc) {                       // poll the other cluster's lines until every tag is this meeting's
                    uint4 q[NQ];
                    bool ok = false;
                    for (unsigned it = 0; it < (1u << 22); ++it) {
                        const uint4 w = ld_line(lsrc + NQ - 1);
                        if (w.y == stage && w.w == stage) break;
                        __nanosleep(it < 64 ? 20 : 200);
                    }
                    for (unsigned it = 0; it < (1u << 20) && !ok; ++it) {
#pragma unroll
                        for (int j = 0; j < NQ; ++j) q[j] = ld_line(lsrc + j);
                        ok = true;
#pragma unroll
                        for (int j = 0; j < NQ; ++j) ok = ok && q[j].y == stage && q[j].w == stage;
                        if (!ok) __nanosleep(100);
                    }
                    if (!ok) atomicExch(fault, 1u);
#pragma unroll
                    for (int j = 0; j < NQ; ++j) Line<T>::get(q[j], &v[j * Line<T>::per]);
                }
                __syncwarp();
            }
            parity ^= 1;
        }
    };
    auto meet = [&]() {
        if constexpr (CL) { meet_cluster(); return; }
        if (a.sync_mode == kSyncLL) { meet_lines(); return; }
        // publish the outermost valid lanes, meet the neighbours, refresh the halo lanes
        ++stage;
        if (active) {
            T* mine = xbuf + ((size_t)parity * a.ntiles + tile) * 2 * side;
            if (own_l || own_r) {
                T* dst = mine + (own_l ? (size_t)(lane - hl) * C : side + (size_t)(lane - (32 - 2 * hl)) * C);
#pragma unroll
                for (int j = 0; j < C / V; ++j) {
                    T t[V];
#pragma unroll
                    for (int i = 0; i < V; ++i) t[i] = v[j * V + i];
                    st_vec_cg(dst + j * V, t);
                }
            }
        }
        signal();
        await();
        if (active) {
            const T* src = nullptr;
            if (halo_l && has_l)      // the left neighbour's right side
                src = xbuf + ((size_t)parity * a.ntiles + tile - 1) * 2 * side + side + (size_t)lane * C;
            else if (halo_r && has_r) // the right neighbour's left side
                src = xbuf + ((size_t)parity * a.ntiles + tile + 1) * 2 * side + (size_t)(lane - (32 - hl)) * C;
            if (src) {
#pragma unroll
                for (int j = 0; j < C / V; ++j) {
                    T t[V];
                    ld_vec_cg(src + j * V, t);
#pragma unroll
                    for (int i = 0; i < V; ++i) v[j * V + i] = t[i];
                }
            }
        }
        parity ^= 1;
    };

    if (a.sync_mode == kSyncStagger) {
        // Staggered flag-in-data meetings.  Every tile publishes its edge lanes every tb/2 levels, but refreshes
        // its own halo only every second time: the two CTAs that share an SM take opposite turns (the turn is
        // the order in which they arrived on the SM), so while one warp of a scheduler waits for its neighbours'
        // lines the other one computes.  Any assignment of turns is correct -- a tile only ever reads lines of
        // the level it is at.
        __shared__ int turn_s;
        if (threadIdx.x == 0) {
            unsigned smid;
            asm volatile("mov.u32 %0, %%smid;" : "=r"(smid));
            turn_s = (int)(atomicAdd(flags + a.ntiles + 1 + (smid & 255u), 1u) & 1u);
        }
        __syncthreads();
        const int turn = turn_s;
        const int tbh = a.tb / 2 - (a.tb / 2) % 2;             // levels between two publications (even)
        int64_t left = a.steps;
        int usedh = 0, h = 0;
        auto half = [&]() {
            const unsigned tag = a.epoch0 + 1 + (unsigned)h;
            publish_lines(h & (kLineSlots - 1), tag);
            if ((h & 1) != turn) consume_lines(h & (kLineSlots - 1), tag);
            ++h; usedh = 0;
        };
        if (a.phase0 == 0 && left > 0) { level_I<T, C, false>(v, c, 0); usedh = 2; --left; }
#pragma unroll 1
        while (left >= 2) {
            if (usedh + 2 > tbh) half();
            level_R<T, C, false>(v, x0, c, 0);
            level_L<T, C, false>(v, x0, c, 0);
            usedh += 2; left -= 2;
        }
        if (left) {
            if (usedh + 2 > tbh) half();
            level_R<T, C, false>(v, x0, c, 0);
            unshift<T, C, false>(v, x0, c, 0);
        }
        {   // before u is overwritten every neighbour must have loaded it: one last exchange that everybody consumes
            const unsigned tag = a.epoch0 + 1 + (unsigned)h;
            publish_lines(h & (kLineSlots - 1), tag);
            consume_lines(h & (kLineSlots - 1), tag);
        }
        if (inside && lane >= hl && lane < 32 - hl) {
#pragma unroll
            for (int j = 0; j < C / V; ++j) {
                T t[V];
#pragma unroll
                for (int i = 0; i < V; ++i) t[i] = v[j * V + i];
                st_vec(u + e0 + j * V, t);
            }
        }
        return;
    }

    int64_t left = a.steps;
    int usedl = 0;
    if (a.phase0 == 0 && left > 0) { level_I<T, C, false>(v, c, 0); usedl = 2; --left; }
#pragma unroll 1
    while (left >= 2) {
        if (usedl + 2 > a.tb) { meet(); usedl = 0; }
        // two level pairs back to back where the halo allows it: the scheduler overlaps the tail of one
        // pair with the head of the next (a lone warp drains its pipeline at every loop back-edge)
        // (not for the largest tiles: their window alone takes half the register file)
        if constexpr (C * sizeof(T) <= 256) {
            if (left >= 4 && usedl + 4 <= a.tb) {
                level_R<T, C, false>(v, x0, c, 0);
                level_L<T, C, false>(v, x0, c, 0);
                level_R<T, C, false>(v, x0, c, 0);
                level_L<T, C, false>(v, x0, c, 0);
                usedl += 4; left -= 4;
                continue;
            }
        }
        level_R<T, C, false>(v, x0, c, 0);
        level_L<T, C, false>(v, x0, c, 0);
        usedl += 2; left -= 2;
    }
    if (left) {
        if (usedl + 2 > a.tb) { meet(); usedl = 0; }
        level_R<T, C, false>(v, x0, c, 0);
        unshift<T, C, false>(v, x0, c, 0);
    }
    // with no meeting at all the neighbours may still be reading u: wait for their stage 0 (flags), or
    // hold one meeting whose lines can only arrive from a neighbour that has loaded (flag-in-data)
    if (stage == a.epoch0 + 1) { if (a.sync_mode == kSyncLL) meet_lines(); else await(); }
    if (inside && lane >= hl && lane < 32 - hl) {
#pragma unroll
        for (int j = 0; j < C / V; ++j) {
            T t[V];
#pragma unroll
            for (int i = 0; i < V; ++i) t[i] = v[j * V + i];
            st_vec(u + e0 + j * V, t);
        }
    }
    // a CTA's shared memory must outlive its neighbours' reads of it
    if constexpr (CL) cg::this_cluster().sync();
}

}  // namespace ge
