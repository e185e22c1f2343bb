// ge_stream.cuh -- strategy B (1-D), the HBM-streaming form: tb levels per HBM
// round trip with TMA-staged tiles.
//
// The warp-per-tile kernel of ge_temporal.cuh loads each lane's C consecutive
// values straight from global memory: a warp-wide 16-byte load then touches 32
// different 128-byte lines, and the L1 tag stage (not HBM) sets the pace --
// measured on C4: 1.08 ms per launch whatever tb, against 0.66 ms of HBM time.
// Here the tile travels as ONE bulk copy (cp.async.bulk, the TMA engine, no LSU
// involvement) into shared memory, the lanes pick their chunks up from there,
// and the result goes back the same way:
//
//   * a warp is an independent pipeline over its tiles (persistent grid, static
//     round-robin): while it computes tile i from registers, the bulk load of
//     tile i+1 is in flight into the warp's second buffer, and the bulk store of
//     tile i-1 drains from it.  Two buffers and two mbarriers per warp; no
//     __syncthreads anywhere.
//   * a lane's chunk is C values with C*sizeof(T) = 144, 176 or 208 bytes (C =
//     18, 22, 26 fp64; 36, 44, 52 fp32): the lane stride is an odd multiple of 16 bytes, so the 16-byte
//     shared-memory accesses of a quarter-warp fall into 8 different bank
//     groups -- conflict-free without padding, and the tile stays ONE linear
//     block (5632 bytes at the default C) that a single 1-D bulk copy moves.
//   * tile layout, level code and arithmetic are those of the drift-free
//     warp-per-tile kernel (ge_temporal.cuh temporal1d_tile_df; level code in
//     ge_resident.cuh): tile 0 left-aligned, last tile right-aligned, tb stale
//     nodes per side in between.  Bit-identical results.
#pragma once
#include "ge_common.cuh"
#include "ge_resident.cuh"
#include "ge_temporal.cuh"

namespace ge {

constexpr int kStreamWarps = 4;

__device__ __forceinline__ uint32_t smem_u32(const void* p) {
    return (uint32_t)__cvta_generic_to_shared(p);
}
__device__ __forceinline__ void mbar_init(uint64_t* bar, uint32_t count) {
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(smem_u32(bar)), "r"(count) : "memory");
}
__device__ __forceinline__ void mbar_expect_tx(uint64_t* bar, uint32_t bytes) {
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(smem_u32(bar)), "r"(bytes) : "memory");
}
__device__ __forceinline__ void mbar_wait(uint64_t* bar, uint32_t parity) {
    asm volatile(
        "{\n"
        ".reg .pred p;\n"
        "WAIT_%=:\n"
        "mbarrier.try_wait.parity.shared::cta.b64 p, [%0], %1;\n"
        "@p bra DONE_%=;\n"
        "bra WAIT_%=;\n"
        "DONE_%=:\n"
        "}\n" ::"r"(smem_u32(bar)), "r"(parity) : "memory");
}
// global -> shared bulk copy (TMA), completion counted in bytes on the mbarrier
__device__ __forceinline__ void bulk_load(void* smem_dst, const void* gmem_src, uint32_t bytes, uint64_t* bar) {
    asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];"
                 ::"r"(smem_u32(smem_dst)), "l"(gmem_src), "r"(bytes), "r"(smem_u32(bar)) : "memory");
}
// shared -> global bulk copy (TMA), tracked by the bulk async-group
__device__ __forceinline__ void bulk_store(void* gmem_dst, const void* smem_src, uint32_t bytes) {
    asm volatile("cp.async.bulk.global.shared::cta.bulk_group [%0], [%1], %2;"
                 ::"l"(gmem_dst), "r"(smem_u32(smem_src)), "r"(bytes) : "memory");
    asm volatile("cp.async.bulk.commit_group;" ::: "memory");
}
__device__ __forceinline__ void bulk_wait_read() { asm volatile("cp.async.bulk.wait_group.read 0;" ::: "memory"); }
__device__ __forceinline__ void bulk_wait_all() { asm volatile("cp.async.bulk.wait_group 0;" ::: "memory"); }
__device__ __forceinline__ void fence_async_smem() { asm volatile("fence.proxy.async.shared::cta;" ::: "memory"); }

template <typename T>
__device__ __forceinline__ void lds_vec(const T* p, T (&x)[VecOf<T>::V]) {
    using VT = typename VecOf<T>::type;
    const VT v = *reinterpret_cast<const VT*>(p);
    if constexpr (VecOf<T>::V == 4) { x[0] = v.x; x[1] = v.y; x[2] = v.z; x[3] = v.w; }
    else { x[0] = v.x; x[1] = v.y; }
}

// per-item geometry: item = rod * ntiles + tile
struct StreamItem {
    int64_t rod;
    int64_t a0;        // first element of the loaded window
    int64_t out_lo;    // outputs [out_lo, out_hi)
    int64_t out_hi;
    bool first, last;
};
__device__ __forceinline__ StreamItem stream_item(int64_t item, int64_t nx, int W, const Temporal1dGeom& g,
                                                  const Temporal1dTiles& tl) {
    StreamItem it;
    it.rod = item / tl.ntiles;
    const int64_t tile = item - it.rod * tl.ntiles;
    it.first = tile == 0; it.last = tile == tl.nreg;
    it.a0 = it.first ? 0 : (it.last ? nx - W : tile * g.valid - g.halo);
    it.out_lo = tile * g.valid;
    it.out_hi = it.last ? nx : it.out_lo + g.valid;
    return it;
}

template <typename T, int C, bool BC>
__device__ __forceinline__ void stream_levels(T (&v)[C], const Coef1<T>& k, const Temporal1dGeom& g, bool first,
                                              bool last, int lane) {
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
}

template <typename T, int C>
__global__ void __launch_bounds__(kStreamWarps * 32)
ge1d_stream_kernel(const T* __restrict__ uin, T* __restrict__ uout, int64_t nx, int64_t batch,
                   const Coef1<T>* __restrict__ coef, const Temporal1dGeom g, const Temporal1dTiles tl) {
    constexpr int V = VecOf<T>::V;
    constexpr int W = 32 * C;                          // elements per tile window
    constexpr uint32_t kBytes = W * sizeof(T);
    static_assert((C * sizeof(T)) % 32 == 16, "lane stride must be an odd multiple of 16 bytes");
    extern __shared__ __align__(128) unsigned char smem_raw[];
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    // per warp: two tile buffers, then (after all buffers) two mbarriers
    T* buf0 = reinterpret_cast<T*>(smem_raw) + (size_t)warp * 2 * W;
    uint64_t* bars = reinterpret_cast<uint64_t*>(smem_raw + (size_t)kStreamWarps * 2 * kBytes) + warp * 2;
    if (lane == 0) {
        mbar_init(bars + 0, 1);
        mbar_init(bars + 1, 1);
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    __syncwarp();

    const int64_t items = batch * tl.ntiles;
    const int64_t stride = (int64_t)gridDim.x * kStreamWarps;
    int64_t item = (int64_t)blockIdx.x * kStreamWarps + warp;
    if (item >= items) return;
    StreamItem cur = stream_item(item, nx, W, g, tl);
    if (lane == 0) {
        mbar_expect_tx(bars + 0, kBytes);
        bulk_load(buf0, uin + cur.rod * nx + cur.a0, kBytes, bars + 0);
    }
    for (int i = 0; item < items; ++i, item += stride) {
        const int b = i & 1;
        T* buf = buf0 + (size_t)b * W;
        const int64_t next = item + stride;
        StreamItem nxt = cur;
        if (next < items) {
            nxt = stream_item(next, nx, W, g, tl);
            if (lane == 0) {
                bulk_wait_read();                          // the store of item i-1 has left the other buffer
                mbar_expect_tx(bars + (b ^ 1), kBytes);
                bulk_load(buf0 + (size_t)(b ^ 1) * W, uin + nxt.rod * nx + nxt.a0, kBytes, bars + (b ^ 1));
            }
        }
        mbar_wait(bars + b, (uint32_t)((i >> 1) & 1));
        T v[C];
        T* mine = buf + lane * C;
#pragma unroll
        for (int c = 0; c < C / V; ++c) {
            T t[V];
            lds_vec(mine + c * V, t);
#pragma unroll
            for (int j = 0; j < V; ++j) v[c * V + j] = t[j];
        }
        const Coef1<T> k = coef[cur.rod];
        if (cur.first || cur.last) stream_levels<T, C, true>(v, k, g, cur.first, cur.last, lane);
        else                       stream_levels<T, C, false>(v, k, g, false, false, lane);
#pragma unroll
        for (int c = 0; c < C / V; ++c) {
            T t[V];
#pragma unroll
            for (int j = 0; j < V; ++j) t[j] = v[c * V + j];
            using VT = typename VecOf<T>::type;
            VT q;
            if constexpr (V == 4) { q.x = t[0]; q.y = t[1]; q.z = t[2]; q.w = t[3]; } else { q.x = t[0]; q.y = t[1]; }
            *reinterpret_cast<VT*>(mine + c * V) = q;
        }
        fence_async_smem();                                // generic-proxy writes -> visible to the TMA engine
        __syncwarp();
        if (lane == 0)
            bulk_store(uout + cur.rod * nx + cur.out_lo, buf + (cur.out_lo - cur.a0),
                       (uint32_t)((cur.out_hi - cur.out_lo) * sizeof(T)));
        cur = nxt;
    }
    if (lane == 0) bulk_wait_all();
}

template <typename T, int C>
inline size_t stream_smem_bytes() { return (size_t)kStreamWarps * 2 * 32 * C * sizeof(T) + kStreamWarps * 2 * sizeof(uint64_t); }

// Host launcher: tb levels starting at a level of the given phase, persistent grid of `ctas` CTAs.
// Requires nx % V == 0, nx >= 32*C, 16-byte aligned rows.
template <typename T, int C>
inline cudaError_t stream1d_launch(const T* uin, T* uout, int64_t nx, int64_t batch, const Coef1<T>* coef, int tb,
                                   int phase, int ctas, cudaStream_t s) {
    const Temporal1dGeom g = temporal1d_geom(C, VecOf<T>::V, tb, phase);
    const Temporal1dTiles tl = temporal1d_tiles(C, g, nx);
    const int64_t items = batch * tl.ntiles;
    int64_t need = (items + kStreamWarps - 1) / kStreamWarps;
    if (need > ctas) need = ctas;
    ge1d_stream_kernel<T, C><<<(unsigned)need, kStreamWarps * 32, stream_smem_bytes<T, C>(), s>>>(
        uin, uout, nx, batch, coef, g, tl);
    return cudaGetLastError();
}

}  // namespace ge
