// ge_unit_k.cuh -- strategy B for the paper's general scheme (sub-domain length k >= 2) with
// the state in REGISTERS: tb levels per HBM round trip, a thread holds 2k consecutive nodes for all of them.
//
// ge1d_temporal_k_kernel keeps the window in shared memory because the unit grid shifts by k between levels
// (PAPER.md:92, :148); it ends up bound by shared-memory wavefronts (one 8-byte read and write per node update,
// profiles/r02_c4_temporal_k16_ncu.md).  The shift does not force that.  Let a thread hold the nodes
// 2km+1 .. 2km+2k -- the unit-grid cell moved up by one node, window positions p = 0 .. 2k-1.  Then
//   phase 0 (class c = p+1 mod 2k): the confluence pair (c = 2k-1, 0) sits at p = 2k-2, 2k-1 -- both members and
//     three of its four old inputs are the thread's own, the fourth (old node p = 0 of the next lane) it received
//     one level earlier; the A sweep (Eq (1), ascending) runs over p = 0 .. k-2 starting from the PREVIOUS lane's new
//     right pair member, the B sweep (Eq (2), descending) over p = 2k-3 .. k-1 starting from the own left member;
//   phase 1 (c = p+1-k mod 2k): the pair sits at p = k-2, k-1, entirely own; A runs up over p = k .. 2k-2, B down
//     over p = k-3 .. 0 and ends on the previous lane's p = 2k-1, i.e. the thread finishes the NEXT lane's B sweep
//     on its own last node.
// Per level ONE value crosses a lane boundary (phase 0: the new right pair member goes up a lane; phase 1: the end
// of the B chain goes down a lane), and what was received doubles as the old-level input the following level needs
// from that neighbour.  Inside a warp that is one shuffle; between the warps of a CTA one shared-memory word and one
// __syncthreads per level.  Everything else is register arithmetic with compile-time indices: 3 floating-point
// instructions per node update, as in the k = 1 kernels.
// No boundary logic: the CTA's tile carries halo lanes (what an end of the tile spoils moves inward by <= k+1 nodes
// per level), and the two ends of the ROD, where the Dirichlet nodes cut units and sweeps, are recomputed afterwards
// by ge1d_temporal_k_kernel on two windows (ge_api.cu).  Same expressions on the same operands as the per-level
// kernel: bit-identical.
#pragma once
#include "ge_common.cuh"

namespace ge {

#ifndef GE_UNIT_WARPS
#define GE_UNIT_WARPS 8
#endif
#ifndef GE_UNIT_MINB
#define GE_UNIT_MINB 3
#endif
constexpr int kUnitWarps = GE_UNIT_WARPS;         // warps of a CTA = one tile of 32 * kUnitWarps units

struct UnitKGeom {
    int halo_lanes;        // units per side of a tile that are not stored
    int valid_lanes;       // 32 * kUnitWarps - 2 * halo_lanes
    int64_t tiles;         // CTAs per rod
};
inline UnitKGeom unit_k_geom(int k, int tb, int64_t nx) {
    UnitKGeom g;
    g.halo_lanes = (tb * (k + 1) + 2 * k - 1) / (2 * k) + 1;
    g.valid_lanes = 32 * kUnitWarps - 2 * g.halo_lanes;
    const int64_t units = (nx + 2 * k - 1) / (2 * (int64_t)k);
    g.tiles = g.valid_lanes > 0 ? (units + g.valid_lanes - 1) / g.valid_lanes : 0;
    return g;
}

// elements of padding per lane row in shared memory: the row stride must be an odd multiple of 16 bytes
template <typename T, int K> struct UnitPad {
    static constexpr int V = 16 / (int)sizeof(T);
    static constexpr int chunks = 2 * K / V;                       // 16-byte chunks per lane
    static constexpr int pad = (chunks % 2 == 1) ? 0 : V;
    static constexpr int stride = 2 * K + pad;                     // elements
};

// Saul'yev node with its new-level neighbour `chain` (Eq (1): the node below; Eq (2): the node above) and the old
// value `other` of its other neighbour -- ge_level_k.cuh's expression
template <typename T>
__device__ __forceinline__ T sweep_node(T chain, T old, T other, T e) { return fma(e, (chain - old) + (other - old), old); }

// value of lane (tid + DIR) of the CTA: a shuffle inside the warp, a shared-memory word (double-buffered by the
// level's parity, one __syncthreads) between warps.  The end lanes of the CTA get their own value (halo).
template <typename T, int DIR>
__device__ __forceinline__ T unit_neighbour(T x, T* __restrict__ edge, int par, int lane, int warp) {
    constexpr unsigned FULL = 0xffffffffu;
    T* line = edge + par * (2 * kUnitWarps);
    if (DIR < 0) { if (lane == 31) line[warp] = x; } else { if (lane == 0) line[kUnitWarps + warp] = x; }
    __syncthreads();
    T y = DIR < 0 ? __shfl_up_sync(FULL, x, 1) : __shfl_down_sync(FULL, x, 1);
    if (DIR < 0) { if (lane == 0 && warp > 0) y = line[warp - 1]; }
    else         { if (lane == 31 && warp + 1 < kUnitWarps) y = line[kUnitWarps + warp + 1]; }
    return y;
}

template <typename T, int K>
__device__ __forceinline__ void unit_level_p0(T (&v)[2 * K], T& from_prev, const T from_next, T r, T g, T e,
                                              T* __restrict__ edge, int par, int lane, int warp) {
    constexpr int U = 2 * K;
    // the pair (p = U-2, U-1): old inputs v[U-3], v[U-2], v[U-1] and the next lane's old v[0]
    T lo, hi;
    pair_update(v[U - 3], v[U - 2], v[U - 1], from_next, r, g, lo, hi);
    from_prev = unit_neighbour<T, -1>(hi, edge, par, lane, warp);    // the previous lane's new right pair member
    const T saveA = v[K - 1], saveB = v[K - 2];
    T chain = from_prev;
#pragma unroll
    for (int p = 0; p <= K - 2; ++p) {
        const T nxt = p + 1 == K - 1 ? saveA : v[p + 1 < U ? p + 1 : 0];
        chain = sweep_node(chain, v[p], nxt, e);
        v[p] = chain;
    }
    chain = lo;
#pragma unroll
    for (int p = U - 3; p >= K - 1; --p) {
        const T prv = p - 1 == K - 2 ? saveB : v[p - 1 >= 0 ? p - 1 : 0];
        chain = sweep_node(chain, v[p], prv, e);
        v[p] = chain;
    }
    v[U - 2] = lo; v[U - 1] = hi;
}

template <typename T, int K>
__device__ __forceinline__ void unit_level_p1(T (&v)[2 * K], const T from_prev, T& from_next, T r, T g, T e,
                                              T* __restrict__ edge, int par, int lane, int warp) {
    constexpr int U = 2 * K;
    // the pair (p = K-2, K-1): old inputs v[K-3] (K = 2: the previous lane's old last node), v[K-2], v[K-1], v[K]
    T lo, hi;
    pair_update(K >= 3 ? v[K >= 3 ? K - 3 : 0] : from_prev, v[K - 2], v[K - 1], v[K], r, g, lo, hi);
    const T saveC = v[U - 2], last = v[U - 1];
    T chain = hi;
#pragma unroll
    for (int p = K; p <= U - 2; ++p) {
        chain = sweep_node(chain, v[p], v[p + 1], e);
        v[p] = chain;
    }
    chain = lo;
#pragma unroll
    for (int p = K - 3; p >= 0; --p) {
        const T prv = p >= 1 ? v[p >= 1 ? p - 1 : 0] : from_prev;
        chain = sweep_node(chain, v[p], prv, e);
        v[p] = chain;
    }
    v[K - 2] = lo; v[K - 1] = hi;
    // the next lane's B chain ends on this lane's last node
    from_next = unit_neighbour<T, +1>(chain, edge, par, lane, warp);
    v[U - 1] = sweep_node(from_next, last, saveC, e);
    // what the next lane holds at its p = 0 after this level is the end of its chain: K >= 3 its new v[0], K = 2 its lo
}

template <typename T, int K>
__global__ void __launch_bounds__(32 * kUnitWarps, GE_UNIT_MINB)
ge1d_unit_k_kernel(const T* __restrict__ uin, T* __restrict__ uout, int64_t nx, const Coef1<T>* __restrict__ coef,
                   const UnitKGeom g, int phase0, int levels) {
    constexpr int U = 2 * K, V = UnitPad<T, K>::V, CPL = UnitPad<T, K>::chunks, S = UnitPad<T, K>::stride;
    constexpr int L = 32 * kUnitWarps;
    using VT = typename VecOf<T>::type;
    extern __shared__ __align__(16) unsigned char unitk_smem[];
    T* rows = reinterpret_cast<T*>(unitk_smem);                 // L rows of S elements
    T* edge = rows + (size_t)L * S;                              // 2 parities x 2 directions x warps
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const int64_t rod = blockIdx.y;
    const Coef1<T> c = coef[rod];
    const T* __restrict__ in = uin + rod * nx;
    T* __restrict__ out = uout + rod * nx;
    const int64_t unit0 = (int64_t)blockIdx.x * g.valid_lanes - g.halo_lanes;   // unit of thread 0
    const int64_t e0 = unit0 * U;                                               // its first element

    // ---- tile -> shared memory (padded rows), 16-byte chunks, all copies of a thread in flight ----
#pragma unroll
    for (int i = 0; i < CPL; ++i) {
        const int q = i * L + tid;                              // chunk of the tile
        const int64_t el = e0 + (int64_t)q * V;
        T* dst = rows + (q / CPL) * S + (q % CPL) * V;
        if (el >= 0 && el + V <= nx) {
            const uint32_t d32 = (uint32_t)__cvta_generic_to_shared(dst);
            asm volatile("cp.async.cg.shared.global [%0], [%1], 16;" ::"r"(d32), "l"(in + el) : "memory");
        } else {
            VT z;
            if constexpr (V == 4) { z.x = T(0); z.y = T(0); z.z = T(0); z.w = T(0); } else { z.x = T(0); z.y = T(0); }
            *reinterpret_cast<VT*>(dst) = z;
        }
    }
    asm volatile("cp.async.wait_all;" ::: "memory");
    __syncthreads();
    T v[U];
#pragma unroll
    for (int i = 0; i < CPL; ++i) {
        const VT q = *reinterpret_cast<const VT*>(rows + tid * S + i * V);
        if constexpr (V == 4) { v[i * V] = q.x; v[i * V + 1] = q.y; v[i * V + 2] = q.z; v[i * V + 3] = q.w; }
        else { v[i * V] = q.x; v[i * V + 1] = q.y; }
    }
    // the old values a first level needs from its neighbours (afterwards they come with the level's own exchange)
    T from_prev = unit_neighbour<T, -1>(v[U - 1], edge, 0, lane, warp);
    T from_next = unit_neighbour<T, +1>(v[0], edge, 1, lane, warp);
    __syncthreads();
#pragma unroll 1
    for (int lev = 0; lev < levels; ++lev) {
        if (((phase0 + lev) & 1) == 0) unit_level_p0<T, K>(v, from_prev, from_next, c.r, c.g, c.e, edge, lev & 1, lane, warp);
        else                            unit_level_p1<T, K>(v, from_prev, from_next, c.r, c.g, c.e, edge, lev & 1, lane, warp);
    }
    // ---- registers -> shared memory -> coalesced 16-byte stores of the valid lanes ----
    __syncthreads();
#pragma unroll
    for (int i = 0; i < CPL; ++i) {
        VT q;
        if constexpr (V == 4) { q.x = v[i * V]; q.y = v[i * V + 1]; q.z = v[i * V + 2]; q.w = v[i * V + 3]; }
        else { q.x = v[i * V]; q.y = v[i * V + 1]; }
        *reinterpret_cast<VT*>(rows + tid * S + i * V) = q;
    }
    __syncthreads();
#pragma unroll
    for (int i = 0; i < CPL; ++i) {
        const int q = i * L + tid;
        const int ln = q / CPL;
        const int64_t el = e0 + (int64_t)q * V;
        if (ln >= g.halo_lanes && ln < L - g.halo_lanes && el >= 0 && el + V <= nx)
            *reinterpret_cast<VT*>(out + el) = *reinterpret_cast<const VT*>(rows + ln * S + (q % CPL) * V);
    }
}

template <typename T, int K>
inline size_t unit_k_smem() { return ((size_t)32 * kUnitWarps * UnitPad<T, K>::stride + 4 * kUnitWarps) * sizeof(T); }

// tb levels (<= the tb the geometry was made for) from a level of phase `phase`; requires 16-byte aligned rows
// (nx % V == 0 when batch > 1)
template <typename T, int K>
inline cudaError_t unit_k_launch(const T* uin, T* uout, int64_t nx, int64_t batch, const Coef1<T>* coef, int tb,
                                 int phase, int levels, cudaStream_t s) {
    const UnitKGeom g = unit_k_geom(K, tb, nx);
    const size_t smem = unit_k_smem<T, K>();
    cudaError_t e = cudaFuncSetAttribute(ge1d_unit_k_kernel<T, K>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
    if (e == cudaSuccess) e = cudaFuncSetAttribute(ge1d_unit_k_kernel<T, K>, cudaFuncAttributePreferredSharedMemoryCarveout, 100);
    if (e != cudaSuccess) return e;
    dim3 grid((unsigned)g.tiles, (unsigned)batch);
    ge1d_unit_k_kernel<T, K><<<grid, 32 * kUnitWarps, smem, s>>>(uin, uout, nx, coef, g, phase, levels);
    return cudaGetLastError();
}

}  // namespace ge
