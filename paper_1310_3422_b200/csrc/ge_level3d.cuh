// ge_level3d.cuh -- strategy A in 3-D: 2x2x2 eight-point groups, one kernel launch
// per level (reading R-3D -- the paper only claims
// "capacity of extension to higher order dimensions").
//
// Group anchors at (1+phase) mod 2 in every axis (shift (1,1,1) between levels);
// in-group links at the new level, out-of-group links at the old level:
//     (1+3r) new_P - r sum_{3 in-group} new_G = R_P := old_P + r sum_{3 out-of-group} (old_O - old_P)
// The 8x8 block (1+3r) I - r Q3 (Q3 = cube graph) is diagonal in the Walsh basis:
// mode m (a sign pattern over the three axes) has eigenvalue 1 + 2r*popcount(m).
// "Value + correction" form, as everywhere in libge:
//     W = WHT(R);  W_m *= c_{popcount(m)} / 8,  c_j = 2rj / (1 + 2rj)  (W_0 = 0);
//     new = R - WHT(W)
// Groups cut by a face, edge or corner of the box keep their interior members; their
// small system (4, 2 or 1 unknowns, boundary in-group neighbours on the right-hand
// side) is solved by elimination -- only the outermost layer of groups takes this path.
// One thread per group, x fastest: a warp reads 64 consecutive nodes of a row.
#pragma once
#include <type_traits>

#include "ge_common.cuh"

namespace ge {

#ifndef GE_L3D_BX
#define GE_L3D_BX 16
#endif
#ifndef GE_L3D_BY
#define GE_L3D_BY 4
#endif
#ifndef GE_L3D_BZ
#define GE_L3D_BZ 2
#endif
#ifndef GE_L3D_MINB
#define GE_L3D_MINB 1
#endif
constexpr int kLevel3dBx = GE_L3D_BX, kLevel3dBy = GE_L3D_BY, kLevel3dBz = GE_L3D_BZ;   // block of groups (sweeps: GE_NVCC_EXTRA)

template <typename T>
__device__ __forceinline__ void wht8(T (&v)[8]) {
#pragma unroll
    for (int s = 1; s < 8; s <<= 1)
#pragma unroll
        for (int i = 0; i < 8; ++i)
            if (!(i & s)) { const T a = v[i], b = v[i | s]; v[i] = a + b; v[i | s] = a - b; }
}

// Group cut by a face, edge or corner: unknowns = interior members,
// (1+3r) x_P - r sum_{interior partners} x_G = R_P + r sum_{boundary partners} beta; solved by elimination
// (SPD, diagonally dominant: no pivoting).  Only the outermost layer of groups comes here.
template <typename T>
__device__ __forceinline__ void truncated_group3d(const T (&R)[8], const bool (&in)[8], const Coef3<T>& k, T (&nw)[8]) {
    T A[8][8], b[8];
    int idx[8], m = 0;
    for (int d = 0; d < 8; ++d) idx[d] = in[d] ? m++ : -1;
    for (int d = 0; d < 8; ++d) {
        if (idx[d] < 0) continue;
        const int row = idx[d];
        for (int q = 0; q < m; ++q) A[row][q] = T(0);
        A[row][row] = T(1) + T(3) * k.r;
        T rhs = R[d];
        for (int ax = 0; ax < 3; ++ax) {
            const int partner = d ^ (1 << ax);
            if (idx[partner] >= 0) A[row][idx[partner]] = -k.r;
            else {
                // the in-group neighbour is a boundary node of face `ax` (low side if this member has bit 1)
                const bool low = (d >> ax) & 1;
                rhs += k.r * (low ? k.lo[ax] : k.hi[ax]);
            }
        }
        b[row] = rhs;
    }
    for (int c = 0; c < m; ++c) {
        for (int rr = c + 1; rr < m; ++rr) {
            const T f = A[rr][c] / A[c][c];
            for (int cc = c; cc < m; ++cc) A[rr][cc] -= f * A[c][cc];
            b[rr] -= f * b[c];
        }
    }
    for (int c = m - 1; c >= 0; --c) {
        T s = b[c];
        for (int cc = c + 1; cc < m; ++cc) s -= A[c][cc] * b[cc];
        b[c] = s / A[c][c];
    }
    for (int d = 0; d < 8; ++d) nw[d] = idx[d] >= 0 ? b[idx[d]] : T(0);
}

// Group cut by exactly ONE face: its four interior members form a 2x2 square in the face's plane,
//   (1+3r) x_P - r (x_P' + x_P'') = R_P + r beta     (P', P'' the in-square partners, beta the face value),
// solved in the Walsh basis of the square like the full group: eigenvalues 1+r, 1+3r (twice), 1+5r,
// x = b - WHT(q . WHT(b)), q = (1 - 1/lambda)/4.  Members ordered j = d_a + 2 d_b, a < b the in-face axes.
// (ge3d_stream_kernel computes the x-cut groups of its rows with the same function: bit-identical.)
template <typename T>
__device__ __forceinline__ void cut4_solve(const T (&R)[4], T r, T beta, T q1, T q2, T q3, T (&x)[4]) {
    T b[4];
#pragma unroll
    for (int j = 0; j < 4; ++j) b[j] = fma(r, beta, R[j]);
    const T s0 = b[0] + b[1], s1 = b[0] - b[1], s2 = b[2] + b[3], s3 = b[2] - b[3];
    const T w0 = (s0 + s2) * q1, w1 = (s1 + s3) * q2, w2 = (s0 - s2) * q2, w3 = (s1 - s3) * q3;
    const T t0 = w0 + w1, t1 = w0 - w1, t2 = w2 + w3, t3 = w2 - w3;
    x[0] = b[0] - (t0 + t2);
    x[1] = b[1] - (t1 + t3);
    x[2] = b[2] - (t0 - t2);
    x[3] = b[3] - (t1 - t3);
}

// the group is cut by the low (the member outside is its first) or high face of axis AX: constant indices only
template <typename T, int AX>
__device__ __forceinline__ void cut4_group3d(const T (&R)[8], bool low, const Coef3<T>& k, T (&nw)[8]) {
    constexpr int A = AX == 0 ? 1 : 0, B = AX == 2 ? 1 : 2;
    T R4[4], x4[4];
#pragma unroll
    for (int j = 0; j < 4; ++j) {
        const int rest = ((j & 1) << A) | ((j >> 1) << B);
        R4[j] = low ? R[rest | (1 << AX)] : R[rest];
    }
    cut4_solve<T>(R4, k.r, low ? k.lo[AX] : k.hi[AX], k.q1, k.q2, k.q3, x4);
#pragma unroll
    for (int j = 0; j < 4; ++j) {
        const int rest = ((j & 1) << A) | ((j >> 1) << B);
        nw[rest | (1 << AX)] = low ? x4[j] : T(0);
        nw[rest] = low ? T(0) : x4[j];
    }
}

// one group, anchored at element (g0, g1, g2)
template <typename T, int PH>
__device__ __forceinline__ void group3d(const T* __restrict__ uin, T* __restrict__ uout, int nx, int ny, int nz,
                                        const Coef3<T>& k, int g0, int g1, int g2) {
    if (g0 >= nx || g1 >= ny || g2 >= nz) return;
    // value of node (x,y,z): interior from memory, one step outside = the face value
    auto val = [&](int x, int y, int z) -> T {
        if (x < 0) return k.lo[0];
        if (x >= nx) return k.hi[0];
        if (y < 0) return k.lo[1];
        if (y >= ny) return k.hi[1];
        if (z < 0) return k.lo[2];
        if (z >= nz) return k.hi[2];
        return __ldg(uin + ((int64_t)z * ny + y) * nx + x);
    };
    const bool full = g0 >= 0 && g0 + 1 < nx && g1 >= 0 && g1 + 1 < ny && g2 >= 0 && g2 + 1 < nz;
    // deep: the group and its 24 out-of-group neighbours are interior nodes -> plain loads at fixed offsets
    const bool deep = g0 >= 1 && g0 + 2 < nx && g1 >= 1 && g1 + 2 < ny && g2 >= 1 && g2 + 2 < nz;
    T R[8];
    bool in[8];
    if (deep) {
        // twelve row pointers (rows y-1 .. y+2 of planes z, z+1; rows y, y+1 of planes z-1, z+2), every load
        // at a constant offset from one of them: the address arithmetic is paid per row, not per load
        const int64_t sy = nx, sz = (int64_t)nx * ny;
        const T* __restrict__ base = uin + ((int64_t)g2 * ny + g1) * nx + g0;
        const T* __restrict__ rp[4][4];
#pragma unroll
        for (int zz = 0; zz < 4; ++zz)
#pragma unroll
            for (int yy = 0; yy < 4; ++yy) rp[zz][yy] = base + (zz - 1) * sz + (yy - 1) * sy;
#pragma unroll
        for (int d = 0; d < 8; ++d) {
            const int dx = d & 1, dy = (d >> 1) & 1, dz = (d >> 2) & 1;
            const T o = __ldg(rp[dz + 1][dy + 1] + dx);
            const T ox = __ldg(rp[dz + 1][dy + 1] + (dx ? 2 : -1));
            const T oy = __ldg(rp[dz + 1][dy ? 3 : 0] + dx);
            const T oz = __ldg(rp[dz ? 3 : 0][dy + 1] + dx);
            in[d] = true;
            R[d] = fma(k.r, ((ox - o) + (oy - o)) + (oz - o), o);
        }
    } else {
#pragma unroll
        for (int d = 0; d < 8; ++d) {
            const int x = g0 + (d & 1), y = g1 + ((d >> 1) & 1), z = g2 + ((d >> 2) & 1);
            in[d] = x >= 0 && x < nx && y >= 0 && y < ny && z >= 0 && z < nz;
            R[d] = T(0);
            if (in[d]) {
                const T o = val(x, y, z);
                const T ox = val(x + ((d & 1) ? 1 : -1), y, z);
                const T oy = val(x, y + ((d & 2) ? 1 : -1), z);
                const T oz = val(x, y, z + ((d & 4) ? 1 : -1));
                R[d] = fma(k.r, ((ox - o) + (oy - o)) + (oz - o), o);
            }
        }
    }
    T nw[8];
    if (full) {
        T W[8];
#pragma unroll
        for (int d = 0; d < 8; ++d) W[d] = R[d];
        wht8(W);
        W[0] = T(0);
        W[1] *= k.c1; W[2] *= k.c1; W[4] *= k.c1;
        W[3] *= k.c2; W[5] *= k.c2; W[6] *= k.c2;
        W[7] *= k.c3;
        wht8(W);
#pragma unroll
        for (int d = 0; d < 8; ++d) nw[d] = R[d] - W[d];
    } else {
        const bool c0 = !(g0 >= 0 && g0 + 1 < nx), c1 = !(g1 >= 0 && g1 + 1 < ny), c2 = !(g2 >= 0 && g2 + 1 < nz);
        if ((int)c0 + (int)c1 + (int)c2 == 1) {
            if (c0)      cut4_group3d<T, 0>(R, g0 < 0, k, nw);
            else if (c1) cut4_group3d<T, 1>(R, g1 < 0, k, nw);
            else         cut4_group3d<T, 2>(R, g2 < 0, k, nw);
        } else {
            truncated_group3d<T>(R, in, k, nw);
        }
    }
    if (full) {
        T* __restrict__ ob = uout + ((int64_t)g2 * ny + g1) * nx + g0;
        const int64_t sy = nx, sz = (int64_t)nx * ny;
        // phase 0: the anchor column is even, a row's two members are one aligned 8- / 16-byte store (nx even)
        const bool pairs = PH == 0 && (nx & 1) == 0 && ((uintptr_t)uout % (2 * sizeof(T))) == 0;
        if (pairs) {
            using P2 = typename std::conditional<sizeof(T) == 8, double2, float2>::type;
#pragma unroll
            for (int d = 0; d < 8; d += 2) {
                P2 v; v.x = nw[d]; v.y = nw[d + 1];
                *reinterpret_cast<P2*>(ob + ((d >> 2) & 1) * sz + ((d >> 1) & 1) * sy) = v;
            }
        } else {
#pragma unroll
            for (int d = 0; d < 8; ++d) ob[((d >> 2) & 1) * sz + ((d >> 1) & 1) * sy + (d & 1)] = nw[d];
        }
    } else {
#pragma unroll
        for (int d = 0; d < 8; ++d)
            if (in[d]) {
                const int x = g0 + (d & 1), y = g1 + ((d >> 1) & 1), z = g2 + ((d >> 2) & 1);
                uout[((int64_t)z * ny + y) * nx + x] = nw[d];
            }
    }
}

constexpr int kLevel3dGy = 1;       // groups per thread, consecutive in y (2 measured: no gain, the register allocation serialises them)

template <typename T, int PH>
__global__ void __launch_bounds__(kLevel3dBx * kLevel3dBy * kLevel3dBz, GE_L3D_MINB)
ge3d_level_kernel(const T* __restrict__ uin, T* __restrict__ uout, int nx, int ny, int nz,
                  const Coef3<T>* __restrict__ coef) {
    const Coef3<T> k = *coef;
    const int g0 = 2 * (blockIdx.x * kLevel3dBx + threadIdx.x) - PH;      // anchor, 0-based element indices
    const int g1 = 2 * kLevel3dGy * (blockIdx.y * kLevel3dBy + threadIdx.y) - PH;
    const int g2 = 2 * (blockIdx.z * kLevel3dBz + threadIdx.z) - PH;
#pragma unroll
    for (int s = 0; s < kLevel3dGy; ++s) group3d<T, PH>(uin, uout, nx, ny, nz, k, g0, g1 + 2 * s, g2);
}

template <typename T>
inline cudaError_t level3d_launch(const T* uin, T* uout, int64_t nx, int64_t ny, int64_t nz, const Coef3<T>* coef,
                                  int phase, cudaStream_t s) {
    auto groups = [&](int64_t n) { return (n + phase) / 2 + 1; };      // anchors -phase, 2-phase, ... <= n-1
    dim3 block(kLevel3dBx, kLevel3dBy, kLevel3dBz);
    dim3 grid((unsigned)((groups(nx) + kLevel3dBx - 1) / kLevel3dBx),
              (unsigned)((groups(ny) + kLevel3dBy * kLevel3dGy - 1) / (kLevel3dBy * kLevel3dGy)),
              (unsigned)((groups(nz) + kLevel3dBz - 1) / kLevel3dBz));
    if (phase == 0) ge3d_level_kernel<T, 0><<<grid, block, 0, s>>>(uin, uout, (int)nx, (int)ny, (int)nz, coef);
    else            ge3d_level_kernel<T, 1><<<grid, block, 0, s>>>(uin, uout, (int)nx, (int)ny, (int)nz, coef);
    return cudaGetLastError();
}

}  // namespace ge
