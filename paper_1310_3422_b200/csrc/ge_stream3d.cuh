// ge_stream3d.cuh -- strategy A in 3-D, streaming form: one level per launch, every thread marches along z.
//
// Scheme: DESIGN.md reading R-3D (2x2x2 eight-point groups anchored at (1+phase) mod 2 in every axis;
// SURVEY.md 8(f) NEXT-4; the paper only claims the extension).  Arithmetic: the
// expression tree of ge_level3d.cuh group3d (right-hand sides, Walsh transform, "value - correction"),
// so the two kernels agree bit for bit.
//
// ge3d_level_kernel gives a thread one group and 32 scalar loads: ~400 issued instructions per group
// against 118 floating-point ones, half of the HBM copy rate.  Here
//   * a lane owns one group COLUMN (two adjacent x nodes, one 8- / 16-byte vector when the anchor column is
//     even) of one group ROW (two y rows) and streams over the group plane pairs of its z segment: the
//     plane below the pair is the previous pair's upper plane, the plane above it the next pair's lower
//     plane -- both already in registers; per group 8 vector loads (4 own, 4 for the rows y-1 and y+2,
//     which the warp above / below loads as its own: L1 / L2 hits), 4 vector stores;
//   * the x neighbours (columns x-1, x+2) are the adjacent lanes' values: 8 shuffles; lanes 0 and 31 fetch
//     theirs with one predicated scalar copy each per row, together with the pair (not when it is needed);
//   * the pairs ahead travel through a lane-private cp.async ring in shared memory (depth 2; deeper rings, a
//     second pair ahead in registers and L2 prefetches were measured and bring nothing: DESIGN.md section 7);
//   * no boundary logic at all: only "deep" groups (the group and its 24 out-of-group neighbours interior,
//     ge_level3d.cuh) are stored; addresses of anything else are clamped into the grid and the results
//     dropped.  The outermost layer of groups -- first and last group index of every axis -- is left to
//     ge3d_shell_kernel, which runs group3d (faces, edges, corners by elimination) on the six faces only.
#pragma once
#include "ge_common.cuh"
#include "ge_level3d.cuh"

namespace ge {

#ifndef GE_S3D_WY
#define GE_S3D_WY 8
#endif
#ifndef GE_S3D_MINB
#define GE_S3D_MINB 2
#endif
#ifndef GE_S3D_UNROLL
#define GE_S3D_UNROLL 1
#endif
constexpr int kS3Unroll = GE_S3D_UNROLL;
#ifndef GE_S3D_WX
#define GE_S3D_WX 1
#endif
constexpr int kS3Wx = GE_S3D_WX;          // warps of a CTA side by side in x (a CTA then reads kS3Wx * 64 consecutive nodes of a row)
constexpr int kS3Wy = GE_S3D_WY;          // ... and stacked in y (their halo rows are each other's own rows)
constexpr int kS3Warps = kS3Wx * kS3Wy;

template <typename T> struct Vec2;
template <> struct Vec2<float>  { using type = float2; };
template <> struct Vec2<double> { using type = double2; };

// the lane's two adjacent x nodes of a row (columns xa, xb = xa + 1 unless clamped at an end of the row);
// VEC: one aligned vector access, else two scalar ones
template <typename T, bool VEC>
__device__ __forceinline__ void ld2(const T* __restrict__ row, int xa, int xb, T (&v)[2]) {
    if constexpr (VEC) {
        const typename Vec2<T>::type q = __ldg(reinterpret_cast<const typename Vec2<T>::type*>(row + xa));
        v[0] = q.x; v[1] = q.y;
    } else { v[0] = __ldg(row + xa); v[1] = __ldg(row + xb); }
}
template <typename T, bool VEC>
__device__ __forceinline__ void st2(T* __restrict__ p, T a, T b) {
    if constexpr (VEC) { typename Vec2<T>::type q; q.x = a; q.y = b; *reinterpret_cast<typename Vec2<T>::type*>(p) = q; }
    else { p[0] = a; p[1] = b; }
}

// one group plane pair as a lane holds it: own[plane][row] = rows y, y+1; halo[plane][0 / 1] = rows y-1 / y+2
// xe[plane][row]: lanes 0 / 31 only -- the column left / right of the warp's 64 (the x neighbour no lane holds)
template <typename T>
struct S3Pair { T own[2][2][2]; T halo[2][2][2]; T xe[2][2]; };

template <typename T, bool VEC>
__device__ __forceinline__ void s3_load_pair(const T* __restrict__ uin, int64_t sz, const int64_t (&ro)[4], int xa,
                                             int xb, int z, int nz, S3Pair<T>& p, bool edge_lane, int xe_col) {
#pragma unroll
    for (int pl = 0; pl < 2; ++pl) {
        int zz = z + pl;
        zz = zz < 0 ? 0 : (zz > nz - 1 ? nz - 1 : zz);
        const T* __restrict__ b = uin + zz * sz;
        ld2<T, VEC>(b + ro[1], xa, xb, p.own[pl][0]);
        ld2<T, VEC>(b + ro[2], xa, xb, p.own[pl][1]);
        ld2<T, VEC>(b + ro[0], xa, xb, p.halo[pl][0]);
        ld2<T, VEC>(b + ro[3], xa, xb, p.halo[pl][1]);
        // with the pair, not when it is needed: a load consumed in the iteration that issues it costs every warp a
        // full memory latency per pair (that is what held the first form of this kernel at half the copy rate)
        if (edge_lane) { p.xe[pl][0] = __ldg(b + ro[1] + xe_col); p.xe[pl][1] = __ldg(b + ro[2] + xe_col); }
    }
}

// ---- the pairs ahead wait in a lane-private shared-memory ring, not in registers ----
// A load that waits in a register is issued where ptxas puts it (it batches or sinks look-ahead loads at will) and
// caps the bytes in flight; cp.async does neither: every thread copies the row vectors of the pair RING-1 ahead
// into its own slots ([slot][vector][thread]: conflict-free, no barrier -- a thread only reads what it copied).
// Slot layout per thread: 8 vectors (own rows y, y+1, halo rows y-1, y+2 of the two planes), then 2 vectors holding
// the four edge values of lanes 0 / 31.
constexpr int kS3SlotVecs = 10;
__device__ __forceinline__ void s3_cp_async(void* smem_dst, const void* gmem_src, int bytes) {
    const uint32_t d = (uint32_t)__cvta_generic_to_shared(smem_dst);
    if (bytes == 16)     asm volatile("cp.async.ca.shared.global [%0], [%1], 16;" ::"r"(d), "l"(gmem_src) : "memory");
    else if (bytes == 8) asm volatile("cp.async.ca.shared.global [%0], [%1], 8;" ::"r"(d), "l"(gmem_src) : "memory");
    else                 asm volatile("cp.async.ca.shared.global [%0], [%1], 4;" ::"r"(d), "l"(gmem_src) : "memory");
}
template <typename T, bool VEC>
__device__ __forceinline__ void s3_request_pair(const T* __restrict__ uin, int64_t sz, const int64_t (&ro)[4], int xa,
                                                int xb, int z, int nz, T* __restrict__ slot, int stride, bool edge_lane,
                                                int xe_col) {
    constexpr int rows[4] = {1, 2, 0, 3};            // own rows y, y+1, then halo rows y-1, y+2
#pragma unroll
    for (int pl = 0; pl < 2; ++pl) {
        int zz = z + pl;
        zz = zz < 0 ? 0 : (zz > nz - 1 ? nz - 1 : zz);
        const T* __restrict__ b = uin + zz * sz;
#pragma unroll
        for (int i = 0; i < 4; ++i) {
            T* dst = slot + (pl * 4 + i) * stride;
            if constexpr (VEC) s3_cp_async(dst, b + ro[rows[i]] + xa, 2 * (int)sizeof(T));
            else { s3_cp_async(dst, b + ro[rows[i]] + xa, (int)sizeof(T)); s3_cp_async(dst + 1, b + ro[rows[i]] + xb, (int)sizeof(T)); }
        }
        if (edge_lane) {
            T* dst = slot + (8 + pl) * stride;
            s3_cp_async(dst, b + ro[1] + xe_col, (int)sizeof(T));
            s3_cp_async(dst + 1, b + ro[2] + xe_col, (int)sizeof(T));
        }
    }
}
template <typename T>
__device__ __forceinline__ void s3_read_pair(const T* __restrict__ slot, int stride, S3Pair<T>& p) {
#pragma unroll
    for (int pl = 0; pl < 2; ++pl) {
#pragma unroll
        for (int i = 0; i < 4; ++i) {
            const typename Vec2<T>::type q = *reinterpret_cast<const typename Vec2<T>::type*>(slot + (pl * 4 + i) * stride);
            if (i < 2) { p.own[pl][i][0] = q.x; p.own[pl][i][1] = q.y; }
            else       { p.halo[pl][i - 2][0] = q.x; p.halo[pl][i - 2][1] = q.y; }
        }
        const typename Vec2<T>::type q = *reinterpret_cast<const typename Vec2<T>::type*>(slot + (8 + pl) * stride);
        p.xe[pl][0] = q.x; p.xe[pl][1] = q.y;
    }
}
__device__ __forceinline__ void s3_commit() { asm volatile("cp.async.commit_group;" ::: "memory"); }
template <int N>
__device__ __forceinline__ void s3_wait() { asm volatile("cp.async.wait_group %0;" ::"n"(N) : "memory"); }

#ifndef GE_S3D_RING_F32
#define GE_S3D_RING_F32 2
#endif
#ifndef GE_S3D_RING_F64
#define GE_S3D_RING_F64 2
#endif
template <typename T> struct S3Ring { static constexpr int n = sizeof(T) == 4 ? GE_S3D_RING_F32 : GE_S3D_RING_F64; };

// RING: pairs of the ring (0: the next pair waits in registers instead).
// Group indices start at 1 in every axis: index 0 and the last one are the shell's.
template <typename T, int PH, bool VEC, int RING>
__global__ void __launch_bounds__(32 * kS3Warps, GE_S3D_MINB)
ge3d_stream_kernel(const T* __restrict__ uin, T* __restrict__ uout, int nx, int ny, int nz,
                   const Coef3<T>* __restrict__ coef, int kseg) {
    constexpr unsigned FULL = 0xffffffffu;
    const int lane = threadIdx.x;
    const int wx = (int)threadIdx.y % kS3Wx, wy = (int)threadIdx.y / kS3Wx;
    const int x0 = 2 * (1 + ((int)blockIdx.x * kS3Wx + wx) * 32 + lane) - PH;   // anchor element of the lane's group column
    const int y0 = 2 * (1 + (int)blockIdx.y * kS3Wy + wy) - PH;
    if (!(y0 + 2 < ny)) return;                                      // the whole warp: its group row is shell or beyond
    const bool deep_x = x0 + 2 < nx;
    const int klast = (nz - 1 + PH) / 2;                             // last group plane pair (shell)
    const int k0 = 1 + (int)blockIdx.z * kseg;
    const int k1 = k0 + kseg < klast ? k0 + kseg : klast;            // deep pairs: 1 .. klast-1
    if (k0 >= k1) return;
    const T r = coef->r, c1 = coef->c1, c2 = coef->c2, c3 = coef->c3;
    const int64_t sy = nx, sz = (int64_t)nx * ny;
    // clamped addressing (only groups that are not deep ever see a clamped address; they are not stored):
    // columns x0, x0+1 clamped one by one, so that a lane next to a clamped one still gets its true neighbour
    // column through the shuffles (vector form: x0 and nx are even, the pair is clamped as a whole to nx-2)
    const int xa = VEC ? (x0 > nx - 2 ? nx - 2 : x0) : (x0 > nx - 1 ? nx - 1 : x0);
    const int xb = x0 + 1 > nx - 1 ? nx - 1 : x0 + 1;
    const int64_t ro[4] = {(int64_t)(y0 - 1) * sy, (int64_t)y0 * sy, (int64_t)(y0 + 1) * sy, (int64_t)(y0 + 2) * sy};
    const int xl = x0 - 1;                                           // lane 0's left / lane 31's right neighbour column
    const int xr = x0 + 2 > nx - 1 ? nx - 1 : x0 + 2;

    extern __shared__ __align__(16) unsigned char s3_smem[];
    const int stride = 2 * 32 * kS3Warps;                            // elements between two vectors of a thread
    T* ring = reinterpret_cast<T*>(s3_smem) + 2 * ((int)threadIdx.y * 32 + lane);
    constexpr int kSlot = kS3SlotVecs * 2 * 32 * kS3Warps;           // elements of one ring slot (all threads)

    T prevU[2][2];                    // rows y, y+1 of the plane below the current pair
    S3Pair<T> cur, nxt;
    {
        const T* __restrict__ b = uin + (int64_t)(2 * k0 - PH - 1) * sz;
        ld2<T, VEC>(b + ro[1], xa, xb, prevU[0]);
        ld2<T, VEC>(b + ro[2], xa, xb, prevU[1]);
    }
    const bool edge_lane = lane == 0 || lane == 31;
    const int xe_col = lane == 0 ? xl : xr;
    s3_load_pair<T, VEC>(uin, sz, ro, xa, xb, 2 * k0 - PH, nz, cur, edge_lane, xe_col);
    int rslot = 0;                    // ring slot of pair k+1
    if constexpr (RING > 0) {
#pragma unroll
        for (int q = 0; q < RING - 1; ++q) {
            s3_request_pair<T, VEC>(uin, sz, ro, xa, xb, 2 * (k0 + 1 + q) - PH, nz, ring + q * kSlot, stride, edge_lane, xe_col);
            s3_commit();
        }
    } else {
        s3_load_pair<T, VEC>(uin, sz, ro, xa, xb, 2 * (k0 + 1) - PH, nz, nxt, edge_lane, xe_col);
    }

    // unrolled by the period of the register rotation (cur <- nxt): no moves
#pragma unroll(kS3Unroll ? 2 : 1)
    for (int k = k0; k < k1; ++k) {
        const int z0 = 2 * k - PH;
        if constexpr (RING > 0) {
            // pair k+RING goes into the slot pair k held (read at the previous iteration); then pair k+1 must have landed
            const int wslot = rslot == 0 ? RING - 1 : rslot - 1;
            s3_request_pair<T, VEC>(uin, sz, ro, xa, xb, z0 + 2 * RING, nz, ring + wslot * kSlot, stride, edge_lane, xe_col);
            s3_commit();
            s3_wait<RING - 1>();
            s3_read_pair<T>(ring + rslot * kSlot, stride, nxt);
            rslot = rslot + 1 == RING ? 0 : rslot + 1;
        }
        // x neighbours of the four rows of the pair: columns x0-1 (left) and x0+2 (right)
        T lf[2][2], rt[2][2];
#pragma unroll
        for (int pl = 0; pl < 2; ++pl)
#pragma unroll
            for (int rr = 0; rr < 2; ++rr) {
                lf[pl][rr] = __shfl_up_sync(FULL, cur.own[pl][rr][1], 1);
                rt[pl][rr] = __shfl_down_sync(FULL, cur.own[pl][rr][0], 1);
            }
#pragma unroll
        for (int pl = 0; pl < 2; ++pl)
#pragma unroll
            for (int rr = 0; rr < 2; ++rr) {
                if (lane == 0) lf[pl][rr] = cur.xe[pl][rr];
                if (lane == 31) rt[pl][rr] = cur.xe[pl][rr];
            }
        // right-hand sides, member d = dx + 2 dy + 4 dz (ge_level3d.cuh group3d)
        T R[8];
#pragma unroll
        for (int d = 0; d < 8; ++d) {
            const int dx = d & 1, dy = (d >> 1) & 1, dz = (d >> 2) & 1;
            const T o = cur.own[dz][dy][dx];
            const T ox = dx ? rt[dz][dy] : lf[dz][dy];
            const T oy = cur.halo[dz][dy][dx];
            const T oz = dz ? nxt.own[0][dy][dx] : prevU[dy][dx];
            R[d] = fma(r, ((ox - o) + (oy - o)) + (oz - o), o);
        }
        T W[8];
#pragma unroll
        for (int d = 0; d < 8; ++d) W[d] = R[d];
        wht8(W);
        W[0] = T(0);
        W[1] *= c1; W[2] *= c1; W[4] *= c1;
        W[3] *= c2; W[5] *= c2; W[6] *= c2;
        W[7] *= c3;
        wht8(W);
        if (deep_x) {
            T* __restrict__ ob = uout + (int64_t)z0 * sz + ro[1] + x0;
#pragma unroll
            for (int dz = 0; dz < 2; ++dz)
#pragma unroll
                for (int dy = 0; dy < 2; ++dy)
                    st2<T, VEC>(ob + dz * sz + dy * sy, R[4 * dz + 2 * dy] - W[4 * dz + 2 * dy],
                                R[4 * dz + 2 * dy + 1] - W[4 * dz + 2 * dy + 1]);
        }
        // slide up by one pair
#pragma unroll
        for (int rr = 0; rr < 2; ++rr) { prevU[rr][0] = cur.own[1][rr][0]; prevU[rr][1] = cur.own[1][rr][1]; }
        cur = nxt;
        if constexpr (RING == 0) s3_load_pair<T, VEC>(uin, sz, ro, xa, xb, z0 + 4, nz, nxt, edge_lane, xe_col);
    }
}

// The outermost layer of groups: first and last group index of every axis.  blockIdx.z = face (axis * 2 + side);
// the face's two other axes are tiled by the block; group3d does faces, edges and corners (by elimination).
// Groups on an edge or corner of the box belong to two or three faces and are written by each with the same value.
template <typename T, int PH>
__global__ void __launch_bounds__(128)
ge3d_shell_kernel(const T* __restrict__ uin, T* __restrict__ uout, int nx, int ny, int nz,
                  const Coef3<T>* __restrict__ coef) {
    const Coef3<T> k = *coef;
    const int n[3] = {nx, ny, nz};
    const int face = blockIdx.z, ax = face >> 1, side = face & 1;
    const int au = ax == 0 ? 1 : 0, av = ax == 2 ? 1 : 2;             // the two in-face axes, au the faster one
    const int last = (n[ax] - 1 + PH) / 2;                            // group index of the last anchor <= n-1
    const int gu = blockIdx.x * 32 + threadIdx.x, gv = blockIdx.y * 4 + threadIdx.y;
    int g[3];
    g[ax] = 2 * (side ? last : 0) - PH;
    g[au] = 2 * gu - PH;
    g[av] = 2 * gv - PH;
    // threads beyond the face fall out inside group3d (anchor >= n)
    group3d<T, PH>(uin, uout, nx, ny, nz, k, g[0], g[1], g[2]);
}

// ge3d_stream_kernel + ge3d_shell_kernel; requires nx even, nx, ny, nz >= 4 and 2-element alignment of both buffers
// for the vector form (otherwise the scalar form is used in phase 0 too)
template <typename T, int PH, bool VEC>
inline cudaError_t stream3d_launch_one(const T* uin, T* uout, int nx, int ny, int nz, const Coef3<T>* coef, int kseg,
                                       dim3 grid, cudaStream_t s) {
    constexpr int RING = S3Ring<T>::n;
    constexpr size_t smem = (size_t)RING * kS3SlotVecs * 2 * 32 * kS3Warps * sizeof(T);
    if (smem > 48 * 1024) {                    // idempotent, a few microseconds against a level of >= 100
        const cudaError_t e = cudaFuncSetAttribute(ge3d_stream_kernel<T, PH, VEC, RING>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
        if (e != cudaSuccess) return e;
    }
    ge3d_stream_kernel<T, PH, VEC, RING><<<grid, dim3(32, kS3Warps), smem, s>>>(uin, uout, nx, ny, nz, coef, kseg);
    return cudaGetLastError();
}

// aux / ev_in / ev_out (optional): the shell kernel runs on the stream `aux`, beside the streaming kernel -- both
// read the old level and write disjoint parts of the new one; ev_in orders it after the work already on `s`,
// ev_out makes `s` wait for it.
template <typename T>
inline cudaError_t stream3d_launch(const T* uin, T* uout, int64_t nx, int64_t ny, int64_t nz, const Coef3<T>* coef,
                                   int phase, int sm_count, cudaStream_t s, cudaStream_t aux = nullptr,
                                   cudaEvent_t ev_in = nullptr, cudaEvent_t ev_out = nullptr) {
    auto last = [&](int64_t n) { return (n - 1 + phase) / 2; };         // group index of the last anchor <= n-1
    const int64_t gx = last(nx) - 1, gy = last(ny) - 1, gz = last(nz) - 1;   // deep groups: indices 1 .. last-1
    auto groups = [&](int64_t n) { return last(n) + 1; };
    const int64_t ax = groups(nx), ay = groups(ny), az = groups(nz);
    const int64_t gmax = ax > ay ? (ax > az ? ax : az) : (ay > az ? ay : az);
    cudaError_t e = cudaSuccess;
    // shell first (it is small and latency-bound: it starts on part of the chip, the streaming kernel fills the rest)
    const bool side = aux && ev_in && ev_out;
    cudaStream_t ss = side ? aux : s;
    if (side) {
        e = cudaEventRecord(ev_in, s);
        if (e == cudaSuccess) e = cudaStreamWaitEvent(aux, ev_in, 0);
        if (e != cudaSuccess) return e;
    }
    dim3 sblock(32, 4), sgrid((unsigned)((gmax + 31) / 32), (unsigned)((gmax + 3) / 4), 6);
    if (phase == 0) ge3d_shell_kernel<T, 0><<<sgrid, sblock, 0, ss>>>(uin, uout, (int)nx, (int)ny, (int)nz, coef);
    else            ge3d_shell_kernel<T, 1><<<sgrid, sblock, 0, ss>>>(uin, uout, (int)nx, (int)ny, (int)nz, coef);
    e = cudaGetLastError();
    if (e != cudaSuccess) return e;
    if (side) { e = cudaEventRecord(ev_out, aux); if (e != cudaSuccess) return e; }
    if (gx > 0 && gy > 0 && gz > 0) {
        // z segments: enough CTAs for ~8 resident CTAs on every SM, at least 8 pairs per segment
        const int64_t bx = (gx + 32 * kS3Wx - 1) / (32 * kS3Wx);
        const int64_t ctas_xy = bx * ((gy + kS3Wy - 1) / kS3Wy);
        int64_t segs = (8 * (int64_t)sm_count + ctas_xy - 1) / ctas_xy;
        if (segs > gz / 8) segs = gz / 8;
        if (segs < 1) segs = 1;
        const int kseg = (int)((gz + segs - 1) / segs);
        dim3 grid((unsigned)bx, (unsigned)((gy + kS3Wy - 1) / kS3Wy), (unsigned)((gz + kseg - 1) / kseg));
        const bool vec = phase == 0 && nx % 2 == 0 && (((uintptr_t)uin | (uintptr_t)uout) % (2 * sizeof(T))) == 0;
        if (phase == 0) e = vec ? stream3d_launch_one<T, 0, true>(uin, uout, (int)nx, (int)ny, (int)nz, coef, kseg, grid, s)
                                : stream3d_launch_one<T, 0, false>(uin, uout, (int)nx, (int)ny, (int)nz, coef, kseg, grid, s);
        else            e = stream3d_launch_one<T, 1, false>(uin, uout, (int)nx, (int)ny, (int)nz, coef, kseg, grid, s);
        if (e != cudaSuccess) return e;
    }
    if (side) e = cudaStreamWaitEvent(s, ev_out, 0);
    return e;
}

}  // namespace ge
