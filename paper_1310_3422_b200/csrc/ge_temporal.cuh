// ge_temporal.cuh -- strategy B (1-D): tb levels per launch, state held in
// registers, one HBM round trip per tb levels.
//
// Blackwell redesign of the paper's synchronisation question (PAPER.md:138-150:
// two block barriers per level pair).  Here a WARP is an independent
// halo-redundant tile: lane t holds C consecutive values; a two-point group
// (i,i+1) reads u_{i-1}..u_{i+2}, so the dependency cone of a
// pair widens by one node per side per level ("one group per sub-step").  The
// warp loads 32*C values, advances tb levels exchanging only two values per
// lane per level through warp shuffles, and stores the 32*C - 2*tb values whose
// cone stayed inside the tile.  No __syncthreads, no shared memory, no
// inter-block barrier: the alternating group shift happens in registers.
//
// Sliding window.  Before a level whose pairs have their left members at odd
// element indices (phase 1), lane t holds elements [a, a+C) with a even.  It
// fetches elements a+C, a+C+1 (the first pair of lane t+1) and updates the pairs
// (a+1,a+2) ... (a+C-1,a+C): its window becomes [a+1, a+C+1).  Now a+1 is odd and
// the next level (phase 0) has its left members at even indices, i.e. again at
// window start + 1: every level is the same code, the window slides right by
// one element per level, and after an even tb it is 16-byte aligned again.
// Hence a temporal block must START AT AN ODD LEVEL (ge_run peels one per-level
// launch if needed) and tb is a multiple of the vector width.
#pragma once
#include "ge_common.cuh"

namespace ge {

template <typename T> struct Temporal1dCfg;
template <> struct Temporal1dCfg<double> { static constexpr int C = 8;  static constexpr int TB = 16; };
template <> struct Temporal1dCfg<float>  { static constexpr int C = 16; static constexpr int TB = 16; };

constexpr int kTemporalWarps = 4;   // warps per CTA (independent tiles)

template <typename T>
inline int temporal1d_round_tb(int64_t tb) {
    constexpr int V = VecOf<T>::V;
    constexpr int C = Temporal1dCfg<T>::C;
    const int64_t maxtb = 8 * C;                 // keeps at least half of the lanes valid
    if (tb > maxtb) tb = maxtb;
    return (int)(tb - tb % V);
}
template <typename T>
inline int temporal1d_pick_tb(int requested) {
    int tb = requested > 0 ? requested : Temporal1dCfg<T>::TB;
    tb = temporal1d_round_tb<T>(tb);
    return tb < VecOf<T>::V ? VecOf<T>::V : tb;
}
template <typename T>
inline int temporal1d_valid_lanes(int tb) {
    constexpr int C = Temporal1dCfg<T>::C;
    return 32 - (2 * tb + C - 1) / C;
}
template <typename T> inline int64_t temporal1d_tile_valid(int tb) { return (int64_t)temporal1d_valid_lanes<T>(tb) * Temporal1dCfg<T>::C; }
template <typename T> inline int64_t temporal1d_tile_loaded() { return 32 * Temporal1dCfg<T>::C; }

template <typename T, int C, bool EDGE>
__device__ __forceinline__ void temporal1d_tile(const T* __restrict__ in, T* __restrict__ out, int64_t nx,
                                                const Coef1<T>& k, int tb, int64_t w_valid,
                                                int64_t tile, int lane) {
    constexpr int V = VecOf<T>::V;
    constexpr unsigned FULL = 0xffffffffu;
    // element index of v[0] before the first level
    const int64_t a0 = tile * w_valid - tb + (int64_t)lane * C;
    T v[C + 2];
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
#pragma unroll 2
    for (int l = 0; l < tb; ++l) {
        v[C] = __shfl_down_sync(FULL, v[0], 1);
        v[C + 1] = __shfl_down_sync(FULL, v[1], 1);
        T nv[C];
#pragma unroll
        for (int m = 0; m < C / 2; ++m) {
            if constexpr (EDGE) {
                const int64_t bidx = a0 + l + 2 * m + 1;    // element index of the pair's left member
                pair_update_bc(v[2 * m], v[2 * m + 1], v[2 * m + 2], v[2 * m + 3], k,
                               bidx == -1, bidx + 1 == nx, nv[2 * m], nv[2 * m + 1]);
            } else {
                pair_update(v[2 * m], v[2 * m + 1], v[2 * m + 2], v[2 * m + 3], k.r, k.g, nv[2 * m], nv[2 * m + 1]);
            }
        }
        if constexpr (EDGE) {
            // keep the Dirichlet ghosts (node 0 = element -1, node N+1 = element nx) constant
#pragma unroll
            for (int j = 0; j < C; ++j) {
                const int64_t idx = a0 + l + 1 + j;
                if (idx == -1) nv[j] = k.lo;
                if (idx == nx) nv[j] = k.hi;
            }
        }
#pragma unroll
        for (int j = 0; j < C; ++j) v[j] = nv[j];
    }
    // window is now [a0 + tb, a0 + tb + C); store the lanes whose cone stayed inside the tile
    const int64_t o0 = tile * w_valid + (int64_t)lane * C;
    if ((int64_t)lane * C < w_valid) {
#pragma unroll
        for (int c = 0; c < C / V; ++c) {
            const int64_t idx = o0 + c * V;
            if (idx + V <= nx) {
                T t[V];
#pragma unroll
                for (int j = 0; j < V; ++j) t[j] = v[c * V + j];
                st_vec(out + idx, t);
            }
        }
    }
}

template <typename T, int C>
__global__ void __launch_bounds__(kTemporalWarps * 32)
ge1d_temporal_kernel(const T* __restrict__ uin, T* __restrict__ uout, int64_t nx, int64_t batch,
                     const Coef1<T>* __restrict__ coef, int tb, int64_t w_valid, int64_t tiles_per_rod) {
    const int lane = threadIdx.x & 31;
    const int warp = threadIdx.x >> 5;
    const int64_t tile = (int64_t)blockIdx.x * kTemporalWarps + warp;
    if (tile >= tiles_per_rod) return;
    for (int64_t rod = blockIdx.y; rod < batch; rod += gridDim.y) {
        const Coef1<T> k = coef[rod];
        const T* __restrict__ in = uin + rod * nx;
        T* __restrict__ out = uout + rod * nx;
        const int64_t lo_idx = tile * w_valid - tb;              // first element touched
        const int64_t hi_idx = lo_idx + 32 * C + tb;             // one past the last element touched
        if (lo_idx < 0 || hi_idx > nx) temporal1d_tile<T, C, true>(in, out, nx, k, tb, w_valid, tile, lane);
        else                           temporal1d_tile<T, C, false>(in, out, nx, k, tb, w_valid, tile, lane);
    }
}

// Host launcher.  Requires: nx % V == 0, 16-byte aligned rows, tb % V == 0, tb >= V,
// and the first of the tb levels is an odd (phase 1) level.  Returns a cudaError_t as int.
template <typename T>
inline int temporal1d_launch(const T* uin, T* uout, int64_t nx, int64_t batch, const Coef1<T>* coef,
                             int tb, cudaStream_t s) {
    constexpr int C = Temporal1dCfg<T>::C;
    const int64_t w_valid = temporal1d_tile_valid<T>(tb);
    const int64_t tiles = (nx + w_valid - 1) / w_valid;
    dim3 grid((unsigned)((tiles + kTemporalWarps - 1) / kTemporalWarps), (unsigned)(batch < 65535 ? batch : 65535));
    ge1d_temporal_kernel<T, C><<<grid, kTemporalWarps * 32, 0, s>>>(uin, uout, nx, batch, coef, tb, w_valid, tiles);
    return (int)cudaGetLastError();
}

}  // namespace ge
