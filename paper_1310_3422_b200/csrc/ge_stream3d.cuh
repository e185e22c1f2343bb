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
//     theirs with one predicated scalar load each per row;
//   * the next pair is loaded while a pair is computed (a second pair ahead, a cp.async ring in shared memory
//     and L2 prefetches were measured and bring nothing: DESIGN.md section 7);
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
constexpr int kS3Wy = GE_S3D_WY;          // warps of a CTA, stacked in y (their halo rows are each other's own rows)

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
template <typename T>
struct S3Pair { T own[2][2][2]; T halo[2][2][2]; };

template <typename T, bool VEC>
__device__ __forceinline__ void s3_load_pair(const T* __restrict__ uin, int64_t sz, const int64_t (&ro)[4], int xa,
                                             int xb, int z, int nz, S3Pair<T>& p) {
#pragma unroll
    for (int pl = 0; pl < 2; ++pl) {
        int zz = z + pl;
        zz = zz < 0 ? 0 : (zz > nz - 1 ? nz - 1 : zz);
        const T* __restrict__ b = uin + zz * sz;
        ld2<T, VEC>(b + ro[1], xa, xb, p.own[pl][0]);
        ld2<T, VEC>(b + ro[2], xa, xb, p.own[pl][1]);
        ld2<T, VEC>(b + ro[0], xa, xb, p.halo[pl][0]);
        ld2<T, VEC>(b + ro[3], xa, xb, p.halo[pl][1]);
    }
}

// Group indices start at 1 in every axis: index 0 and the last one are the shell's.
template <typename T, int PH, bool VEC>
__global__ void __launch_bounds__(32 * kS3Wy, GE_S3D_MINB)
ge3d_stream_kernel(const T* __restrict__ uin, T* __restrict__ uout, int nx, int ny, int nz,
                   const Coef3<T>* __restrict__ coef, int kseg) {
    constexpr unsigned FULL = 0xffffffffu;
    const int lane = threadIdx.x;
    const int x0 = 2 * (1 + (int)blockIdx.x * 32 + lane) - PH;       // anchor element of the lane's group column
    const int y0 = 2 * (1 + (int)blockIdx.y * kS3Wy + (int)threadIdx.y) - PH;
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

    T prevU[2][2];                    // rows y, y+1 of the plane below the current pair
    S3Pair<T> cur, nxt;
    {
        const T* __restrict__ b = uin + (int64_t)(2 * k0 - PH - 1) * sz;
        ld2<T, VEC>(b + ro[1], xa, xb, prevU[0]);
        ld2<T, VEC>(b + ro[2], xa, xb, prevU[1]);
    }
    s3_load_pair<T, VEC>(uin, sz, ro, xa, xb, 2 * k0 - PH, nz, cur);
    s3_load_pair<T, VEC>(uin, sz, ro, xa, xb, 2 * (k0 + 1) - PH, nz, nxt);

    // unrolled by the period of the register rotation (cur <- nxt): no moves
#pragma unroll(kS3Unroll ? 2 : 1)
    for (int k = k0; k < k1; ++k) {
        const int z0 = 2 * k - PH;
        // x neighbours of the four rows of the pair: columns x0-1 (left) and x0+2 (right)
        T lf[2][2], rt[2][2];
#pragma unroll
        for (int pl = 0; pl < 2; ++pl)
#pragma unroll
            for (int rr = 0; rr < 2; ++rr) {
                lf[pl][rr] = __shfl_up_sync(FULL, cur.own[pl][rr][1], 1);
                rt[pl][rr] = __shfl_down_sync(FULL, cur.own[pl][rr][0], 1);
            }
        if (lane == 0 || lane == 31) {
            const T* __restrict__ pa = uin + (int64_t)z0 * sz + (lane == 0 ? xl : xr);
#pragma unroll
            for (int rr = 0; rr < 2; ++rr) {
                const T va = __ldg(pa + ro[1 + rr]);
                const T vb = __ldg(pa + sz + ro[1 + rr]);
                if (lane == 0) { lf[0][rr] = va; lf[1][rr] = vb; } else { rt[0][rr] = va; rt[1][rr] = vb; }
            }
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
        s3_load_pair<T, VEC>(uin, sz, ro, xa, xb, z0 + 4, nz, nxt);
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
    ge3d_stream_kernel<T, PH, VEC><<<grid, dim3(32, kS3Wy), 0, s>>>(uin, uout, nx, ny, nz, coef, kseg);
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
        const int64_t ctas_xy = ((gx + 31) / 32) * ((gy + kS3Wy - 1) / kS3Wy);
        int64_t segs = (8 * (int64_t)sm_count + ctas_xy - 1) / ctas_xy;
        if (segs > gz / 8) segs = gz / 8;
        if (segs < 1) segs = 1;
        const int kseg = (int)((gz + segs - 1) / segs);
        dim3 grid((unsigned)((gx + 31) / 32), (unsigned)((gy + kS3Wy - 1) / kS3Wy), (unsigned)((gz + kseg - 1) / kseg));
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
