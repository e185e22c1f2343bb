// ge_temporal.cuh -- strategy B (1-D): tb levels per launch, state held in
// registers, one HBM round trip per tb levels.
//
// Blackwell redesign of the paper's synchronisation question (PAPER.md:138-150:
// two block barriers per level pair).  Here a WARP is an independent
// halo-redundant tile: lane t holds C consecutive values; a two-point group
// (i,i+1) reads u_{i-1}..u_{i+2} and the pattern shifts by
// one node per level, so a tile edge placed ON a group boundary moves inward by
// one node per level ("one group per sub-step").  The warp loads 32*C values,
// advances tb levels exchanging ONE value per lane per level through a warp
// shuffle, and stores the ~32*C - 2*tb values whose cone stayed inside the
// tile.  No __syncthreads, no shared memory, no inter-block barrier: the
// alternating group shift happens in registers.
//
// Sliding window.  Before a level, lane t holds the window [w, w+C) (element
// indices; element e is node e+1) with the level's left members at w+1, w+3, ...
// It updates the pairs (w+1,w+2) ... (w+C-1,w+C); its window becomes
// [w+1, w+C+1).  The next level's pattern is shifted by one node, i.e. its left
// members again sit at (new window start)+1: every level is the same code and
// the window slides right by one element per level.  A launch that starts at a
// phase-0 level (left members at even elements) first shifts the 16-byte
// aligned window right by one element (`pre`), and after the tb levels the
// window is shifted by `post` < V more elements so that it is 16-byte aligned
// again for the vector stores; each shift is one shuffle per lane.
//
// Arithmetic per level and lane (3 flops per node update; ge_common.cuh has
// the derivation of the factored form).  With e_m = v[2m+1] - v[2m] the
// difference ACROSS the group boundary left of pair m (shared by the two
// adjacent pairs):
//     p_m     = v[2m+1] - r e_m          right-hand side of Eq (2) at the left member
//     z_m     = v[2m]   + r e_m          right-hand side of Eq (1) at the right member
//                                        of the pair to the LEFT (= q_{m-1})
//     q_{C/2-1} comes from lane t+1's z_0 (the one shuffle)
//     w = g (q_m - p_m);  new left = p_m + w;  new right = q_m - w
//
// Interior tiles (no Dirichlet node inside the loaded window -- all but the first and last few)
// take the DRIFT-FREE level code of ge_resident.cuh instead: levels in pairs R/L that slide the
// window right then left, so the state returns to the same registers after two levels (no
// register moves), the halo is symmetric (tb stale nodes on either side) and the tile's output
// range is the same [tile*valid, (tile+1)*valid).  Same expression tree, bit-identical results.
#pragma once
#include "ge_common.cuh"
#include "ge_resident.cuh"

namespace ge {

constexpr int kTemporalWarps = 4;   // warps per CTA (independent tiles)

// Geometry of one launch: fixed by (C, V, tb, starting phase).
struct Temporal1dGeom {
    int tb;        // levels in this launch
    int pre;       // 1 if the launch starts at a phase-0 level
    int post;      // realignment shifts after the last level, < V
    int shift;     // pre + tb + post: element offset between loaded and stored window
    int valid;     // outputs per tile (multiple of V)
    int halo;      // interior tiles: nodes loaded left of the output range (multiple of V, even)
};

inline Temporal1dGeom temporal1d_geom(int C, int V, int tb, int phase) {
    Temporal1dGeom g;
    g.tb = tb;
    g.pre = phase == 0 ? 1 : 0;
    g.post = (V - (g.pre + tb) % V) % V;
    g.shift = g.pre + tb + g.post;
    // a stale slot spreads by 2 slots per level from an even slot, by 3 in the first level from the odd
    // slot the pre-shift leaves behind, by 1 per realignment shift
    const int v = 32 * C - 2 * tb - 2 * g.pre - g.post;
    g.valid = v - v % V;
    // drift-free interior tiles: one stale node per side and level; the in-lane level I that opens a
    // launch at phase 0 and the shift back after an odd number of R/L levels each cost one more
    const int rest = tb - g.pre;
    const int stale = tb + g.pre + (rest & 1);
    g.halo = (stale + V - 1) / V * V;
    if (g.valid > 32 * C - 2 * g.halo) g.valid = 32 * C - 2 * g.halo;
    return g;
}
inline int temporal1d_max_tb(int C) { return 8 * C; }      // keeps at least half of every tile valid

// UA ("unaligned"): rows of any length at any element alignment (batched rods with nx % V != 0, unaligned user
// pointers).  The tile's 32*C elements are read and written with COALESCED scalar accesses -- lane t takes element
// i*32 + t of the window -- and transposed through the warp's own piece of shared memory `sm` (32 rows of C + 1
// elements: conflict-free both ways), so no global access depends on alignment.  Same arithmetic.
template <typename T, int C, bool EDGE, bool UA = false>
__device__ __forceinline__ void temporal1d_tile(const T* __restrict__ in, T* __restrict__ out, int64_t nx,
                                                const Coef1<T>& k, const Temporal1dGeom g,
                                                int64_t tile, int lane, T* __restrict__ sm = nullptr) {
    constexpr int V = VecOf<T>::V;
    constexpr unsigned FULL = 0xffffffffu;
    static_assert(C % 2 == 0 && C % V == 0, "C must hold whole pairs and whole vectors");
    // element index of v[0] at load time
    const int64_t a0 = tile * g.valid - g.shift + (int64_t)lane * C;
    T v[C];
    if constexpr (UA) {
        const int64_t w0 = tile * g.valid - g.shift;                 // the warp's first element
#pragma unroll
        for (int i = 0; i < C; ++i) {
            const int q = i * 32 + lane;
            const int64_t e = w0 + q;
            T x;
            if (!EDGE || (e >= 0 && e < nx)) x = in[e];
            else x = e == -1 ? k.lo : (e == nx ? k.hi : T(0));
            sm[(q / C) * (C + 1) + q % C] = x;
        }
        __syncwarp();
#pragma unroll
        for (int j = 0; j < C; ++j) v[j] = sm[lane * (C + 1) + j];
        __syncwarp();
    } else
#pragma unroll
    for (int c = 0; c < C / V; ++c) {
        const int64_t idx = a0 + c * V;
        T t[V];
        if (!EDGE || (idx >= 0 && idx + V <= nx)) {
            ld_vec(in + idx, t);
        } else {
#pragma unroll
            for (int j = 0; j < V; ++j) t[j] = (idx + j == -1) ? k.lo : ((idx + j == nx) ? k.hi : T(0));
        }
#pragma unroll
        for (int j = 0; j < V; ++j) v[c * V + j] = t[j];
    }
    if (g.pre) shift_window<T, C>(v);
    // EDGE tiles: position of the Dirichlet ghosts relative to the window start, as 32-bit ints
    // (element -1 = node 0, element nx = node N+1); far-away ghosts are clamped out of reach.
    int glo = 0, ghi = 0;
    if constexpr (EDGE) {
        const int64_t w0 = a0 + g.pre;
        const int64_t dlo = -1 - w0, dhi = nx - w0;
        glo = (int)(dlo < -(1 << 20) ? -(1 << 20) : (dlo > (1 << 20) ? (1 << 20) : dlo));
        ghi = (int)(dhi < -(1 << 20) ? -(1 << 20) : (dhi > (1 << 20) ? (1 << 20) : dhi));
    }
    const T r = k.r, gg = k.g;
#pragma unroll 2
    for (int l = 0; l < g.tb; ++l) {
        T p[C / 2], q[C / 2];
        T z0;
#pragma unroll
        for (int m = 0; m < C / 2; ++m) {
            const T e = v[2 * m + 1] - v[2 * m];
            p[m] = fma(-r, e, v[2 * m + 1]);
            const T z = fma(r, e, v[2 * m]);
            if (m == 0) z0 = z; else q[m - 1] = z;
        }
        q[C / 2 - 1] = __shfl_down_sync(FULL, z0, 1);
        T nv[C];
#pragma unroll
        for (int m = 0; m < C / 2; ++m) {
            T pm = p[m], qm = q[m], gm = gg;
            if constexpr (EDGE) {
                // window slot of the pair's left member is 2m+1; slots are relative to w0 + l
                if (2 * m + 1 == glo - l) { pm = k.lo; gm = k.e; }     // left member is node 0
                if (2 * m + 2 == ghi - l) { qm = k.hi; gm = k.e; }     // right member is node N+1
            }
            const T t = qm - pm;
            nv[2 * m] = fma(gm, t, pm);
            nv[2 * m + 1] = fma(-gm, t, qm);
        }
        if constexpr (EDGE) {
            // keep the ghosts constant: new slot j is old slot j+1
#pragma unroll
            for (int j = 0; j < C; ++j) {
                if (j + 1 == glo - l) nv[j] = k.lo;
                if (j + 1 == ghi - l) nv[j] = k.hi;
            }
        }
#pragma unroll
        for (int j = 0; j < C; ++j) v[j] = nv[j];
    }
    for (int s = 0; s < g.post; ++s) shift_window<T, C>(v);
    // window start is now a0 + shift = tile*valid + lane*C: store what stayed inside the cone
    const int64_t o0 = tile * g.valid + (int64_t)lane * C;
    if constexpr (UA) {
#pragma unroll
        for (int j = 0; j < C; ++j) sm[lane * (C + 1) + j] = v[j];
        __syncwarp();
#pragma unroll
        for (int i = 0; i < C; ++i) {
            const int q = i * 32 + lane;
            const int64_t e = tile * g.valid + q;
            if (q < g.valid && e < nx) out[e] = sm[(q / C) * (C + 1) + q % C];
        }
        __syncwarp();
    } else
#pragma unroll
    for (int c = 0; c < C / V; ++c) {
        const int64_t idx = o0 + c * V;
        if (lane * C + c * V < g.valid && idx + V <= nx) {
            T t[V];
#pragma unroll
            for (int j = 0; j < V; ++j) t[j] = v[c * V + j];
            st_vec(out + idx, t);
        }
    }
}

// Drift-free tiles (rods with nx >= 32*C, valid + 2*halo <= 32*C):
//   tile 0            left-aligned: loads [0, 32*C), element 0 in slot 0 of lane 0, writes [0, valid)
//   tile t, 1..nreg-1 loads [t*valid - halo, +32*C) (fits inside the rod), writes [t*valid, (t+1)*valid)
//   tile nreg (last)  right-aligned: loads [nx - 32*C, nx), element nx-1 in slot C-1 of lane 31,
//                     writes [nreg*valid, nx)
// so a Dirichlet node never sits inside a lane and the boundary logic of ge_resident.cuh applies
// (BC = true for the first and last tile only).  nreg*valid <= nx - halo, so the last tile always
// exists, and since tile nreg would not fit, nreg*valid > nx - 32*C + halo: its outputs are valid.
struct Temporal1dTiles {
    int64_t nreg;      // left-aligned + regular tiles
    int64_t ntiles;    // nreg + 1
};
inline Temporal1dTiles temporal1d_tiles(int C, const Temporal1dGeom& g, int64_t nx) {
    Temporal1dTiles t;
    t.nreg = 1 + (nx + g.halo - 32 * (int64_t)C) / g.valid;
    t.ntiles = t.nreg + 1;
    return t;
}

template <typename T, int C, bool BC>
__device__ __forceinline__ void temporal1d_tile_df(const T* __restrict__ in, T* __restrict__ out,
                                                   const Coef1<T>& k, const Temporal1dGeom g, int64_t a0,
                                                   int64_t out_lo, int64_t out_hi, bool first, bool last,
                                                   int lane) {
    constexpr int V = VecOf<T>::V;
    const int64_t e0 = a0 + (int64_t)lane * C;     // element in slot 0 (even: a0, C are)
    T v[C];
#pragma unroll
    for (int c = 0; c < C / V; ++c) {
        T t[V];
        ld_vec(in + e0 + c * V, t);
#pragma unroll
        for (int j = 0; j < V; ++j) v[c * V + j] = t[j];
    }
    ResidentCtx<T, false> cx;
    cx.r = k.r; cx.g = k.g; cx.e = k.e; cx.lo = k.lo; cx.hi = k.hi;
    cx.is_lo = BC && first && lane == 0; cx.is_hi = BC && last && lane == 31;
    cx.lane = lane; cx.warp = 0; cx.nwarps = 1; cx.sx = nullptr;
    T x0 = T(0);
    int left = g.tb;
    if (g.pre) { level_I<T, C, false, BC>(v, cx, 0); --left; }
#pragma unroll 1
    for (; left >= 2; left -= 2) {
        level_R<T, C, false, BC>(v, x0, cx, 0);
        level_L<T, C, false, BC>(v, x0, cx, 0);
    }
    if (left) {
        level_R<T, C, false, BC>(v, x0, cx, 0);
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
ge1d_temporal_kernel(const T* __restrict__ uin, T* __restrict__ uout, int64_t nx, int64_t batch,
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
        if (first || last) temporal1d_tile_df<T, C, true>(in, out, k, g, a0, out_lo, out_hi, first, last, lane);
        else               temporal1d_tile_df<T, C, false>(in, out, k, g, a0, out_lo, out_hi, false, false, lane);
    }
}

// Host launcher: tb levels starting at a level of the given phase.
// Requires nx % V == 0, nx >= 32*C, 16-byte aligned rows, 1 <= tb <= temporal1d_max_tb(C).
template <typename T, int C>
inline cudaError_t temporal1d_launch(const T* uin, T* uout, int64_t nx, int64_t batch, const Coef1<T>* coef,
                                     int tb, int phase, cudaStream_t s) {
    const Temporal1dGeom g = temporal1d_geom(C, VecOf<T>::V, tb, phase);
    const Temporal1dTiles tl = temporal1d_tiles(C, g, nx);
    dim3 grid((unsigned)((tl.ntiles + kTemporalWarps - 1) / kTemporalWarps), (unsigned)(batch < 65535 ? batch : 65535));
    ge1d_temporal_kernel<T, C><<<grid, kTemporalWarps * 32, 0, s>>>(uin, uout, nx, batch, coef, g, tl);
    return cudaGetLastError();
}

template <typename T, int C>
__global__ void __launch_bounds__(kTemporalWarps * 32)
ge1d_temporal_generic_kernel(const T* __restrict__ uin, T* __restrict__ uout, int64_t nx, int64_t batch,
                     const Coef1<T>* __restrict__ coef, const Temporal1dGeom g, int64_t tiles_per_rod) {
    const int lane = threadIdx.x & 31;
    const int warp = threadIdx.x >> 5;
    const int64_t tile = (int64_t)blockIdx.x * kTemporalWarps + warp;
    if (tile >= tiles_per_rod) return;
    const int64_t lo_idx = tile * g.valid - g.shift;          // first element loaded
    const bool edge = lo_idx < 0 || lo_idx + 32 * C > nx;
    for (int64_t rod = blockIdx.y; rod < batch; rod += gridDim.y) {
        const Coef1<T> k = coef[rod];
        const T* __restrict__ in = uin + rod * nx;
        T* __restrict__ out = uout + rod * nx;
        if (edge) temporal1d_tile<T, C, true>(in, out, nx, k, g, tile, lane);
        else      temporal1d_tile<T, C, false>(in, out, nx, k, g, tile, lane);
    }
}

// The same tiles for rows of any length and alignment (temporal1d_tile UA).
template <typename T, int C>
__global__ void __launch_bounds__(kTemporalWarps * 32)
ge1d_temporal_unaligned_kernel(const T* __restrict__ uin, T* __restrict__ uout, int64_t nx, int64_t batch,
                               const Coef1<T>* __restrict__ coef, const Temporal1dGeom g, int64_t tiles_per_rod) {
    __shared__ T sm_all[kTemporalWarps][32 * (C + 1)];
    const int lane = threadIdx.x & 31;
    const int warp = threadIdx.x >> 5;
    const int64_t tile = (int64_t)blockIdx.x * kTemporalWarps + warp;
    if (tile >= tiles_per_rod) return;
    const int64_t lo_idx = tile * g.valid - g.shift;          // first element loaded
    const bool edge = lo_idx < 0 || lo_idx + 32 * C > nx;
    for (int64_t rod = blockIdx.y; rod < batch; rod += gridDim.y) {
        const Coef1<T> k = coef[rod];
        const T* __restrict__ in = uin + rod * nx;
        T* __restrict__ out = uout + rod * nx;
        if (edge) temporal1d_tile<T, C, true, true>(in, out, nx, k, g, tile, lane, sm_all[warp]);
        else      temporal1d_tile<T, C, false, true>(in, out, nx, k, g, tile, lane, sm_all[warp]);
    }
}
// Requires only 1 <= tb <= temporal1d_max_tb(C).
template <typename T, int C>
inline cudaError_t temporal1d_unaligned_launch(const T* uin, T* uout, int64_t nx, int64_t batch, const Coef1<T>* coef,
                                               int tb, int phase, cudaStream_t s) {
    const Temporal1dGeom g = temporal1d_geom(C, VecOf<T>::V, tb, phase);
    const int64_t tiles = (nx + g.valid - 1) / g.valid;
    dim3 grid((unsigned)((tiles + kTemporalWarps - 1) / kTemporalWarps), (unsigned)(batch < 65535 ? batch : 65535));
    ge1d_temporal_unaligned_kernel<T, C><<<grid, kTemporalWarps * 32, 0, s>>>(uin, uout, nx, batch, coef, g, tiles);
    return cudaGetLastError();
}

// Host launcher: tb levels starting at a level of the given phase.
// Requires nx % V == 0, 16-byte aligned rows, 1 <= tb <= temporal1d_max_tb(C).
template <typename T, int C>
inline cudaError_t temporal1d_generic_launch(const T* uin, T* uout, int64_t nx, int64_t batch, const Coef1<T>* coef,
                                     int tb, int phase, cudaStream_t s) {
    const Temporal1dGeom g = temporal1d_geom(C, VecOf<T>::V, tb, phase);
    const int64_t tiles = (nx + g.valid - 1) / g.valid;
    dim3 grid((unsigned)((tiles + kTemporalWarps - 1) / kTemporalWarps), (unsigned)(batch < 65535 ? batch : 65535));
    ge1d_temporal_generic_kernel<T, C><<<grid, kTemporalWarps * 32, 0, s>>>(uin, uout, nx, batch, coef, g, tiles);
    return cudaGetLastError();
}

}  // namespace ge
