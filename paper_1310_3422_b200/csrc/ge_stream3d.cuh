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
//   * every FULL group (all eight nodes in the box) is computed here; a neighbour one step outside the box is the
//     face's value (a select on loop-invariant predicates), addresses of anything else are clamped into the grid
//     and the results dropped.  Groups CUT by a face (anchor -1 in phase 1, anchor n-1) are left to
//     ge3d_shell_kernel, which runs group3d (faces, edges, corners by elimination) on the faces that have cut
//     groups: none in phase 0 and all six in phase 1 when nx, ny, nz are even.
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
#ifndef GE_S3D_MODE
#define GE_S3D_MODE 0
#endif
constexpr int kS3Wx = GE_S3D_WX;          // warps of a CTA side by side in x (a CTA then reads kS3Wx * 64 consecutive nodes of a row)
constexpr int kS3Wy = GE_S3D_WY;          // ... and stacked in y (their halo rows are each other's own rows)
constexpr int kS3Warps = kS3Wx * kS3Wy;

template <typename T> struct Vec2;
template <> struct Vec2<float>  { using type = float2; };
template <> struct Vec2<double> { using type = double2; };

#ifndef GE_S3D_NG_F32
#define GE_S3D_NG_F32 2
#endif
#ifndef GE_S3D_NG_F64
#define GE_S3D_NG_F64 1
#endif
#ifndef GE_S3D_RING_F32
#define GE_S3D_RING_F32 2
#endif
#ifndef GE_S3D_RING_F64
#define GE_S3D_RING_F64 2
#endif
// group columns per lane (a lane's piece of a row is 2*NG nodes: 16 bytes in either precision by default) and
// pairs of the cp.async ring
template <typename T> struct S3Cfg {
    static constexpr int ng = sizeof(T) == 4 ? GE_S3D_NG_F32 : GE_S3D_NG_F64;
    static constexpr int ring = sizeof(T) == 4 ? GE_S3D_RING_F32 : GE_S3D_RING_F64;
};

// one plane pair as a lane holds it, E = 2*NG nodes per row: own[plane][row] = rows y, y+1; halo[plane][0 / 1] =
// rows y-1 / y+2.  Lanes 0 / 31 only (the columns next to the warp's 32*E, which no lane holds):
//   xe[plane][row]  column x0-1 (lane 0) or x0+E (lane 31) of the own rows
//   xe2[plane][row] column x0-2 of the own rows, xh[plane][0 / 1] column x0-1 of the halo rows (lane 0, shifted form)
template <typename T, int E>
struct S3Pair { T own[2][2][E]; T halo[2][2][E]; T xe[2][2]; T xe2[2][2]; T xh[2][2]; };

__device__ __forceinline__ void s3_cp_async(void* smem_dst, const void* gmem_src, int bytes) {
    const uint32_t d = (uint32_t)__cvta_generic_to_shared(smem_dst);
    if (bytes == 16)     asm volatile("cp.async.ca.shared.global [%0], [%1], 16;" ::"r"(d), "l"(gmem_src) : "memory");
    else if (bytes == 8) asm volatile("cp.async.ca.shared.global [%0], [%1], 8;" ::"r"(d), "l"(gmem_src) : "memory");
    else                 asm volatile("cp.async.ca.shared.global [%0], [%1], 4;" ::"r"(d), "l"(gmem_src) : "memory");
}
__device__ __forceinline__ void s3_commit() { asm volatile("cp.async.commit_group;" ::: "memory"); }
template <int N>
__device__ __forceinline__ void s3_wait() { asm volatile("cp.async.wait_group %0;" ::"n"(N) : "memory"); }

// ---- the pairs ahead wait in a lane-private shared-memory ring, not in registers ----
// A load that waits in a register is issued where ptxas puts it (it batches or sinks look-ahead loads at will) and
// caps the bytes in flight; cp.async does neither: every thread copies the row pieces of the pair RING-1 ahead into
// its own slots (conflict-free, no barrier -- a thread only reads what it copied).
// A ring slot: 8 pieces of E nodes per thread ([piece][thread]: own rows y, y+1, halo rows y-1, y+2 of the two
// planes), then kS3Edge values for each of the two edge lanes of every warp ([warp][lane 0 / 31][plane*6 + i]:
// i = 0..3: columns x0-2, x0-1 of own row y, then of y+1 (lane 31: x0+E at i = 1, 3); i = 4, 5: column x0-1 of
// the halo rows).
constexpr int kS3Edge = 12;
template <typename T, int E> struct S3Slot {
    static constexpr int pieces = 8 * E * 32 * kS3Warps;               // elements
    static constexpr int elems = pieces + kS3Warps * 2 * kS3Edge;
};

// xc[e]: column of the lane's node e, clamped into the row one by one (so that a lane next to a clamped one still
// gets its true neighbour column through the shuffles); VEC: xc[0] is 16-byte aligned and the piece contiguous.
// SHIFT: the shifted form's edge values (lane 0: two columns of the own rows, one of the halo rows; lane 31: none).
template <typename T, int E, bool VEC, bool SHIFT>
__device__ __forceinline__ void s3_request_pair(const T* __restrict__ uin, int64_t sz, const int64_t (&ro)[4],
                                                const int (&xc)[E], int z, int nz, T* __restrict__ slot,
                                                T* __restrict__ eslot, int stride, int lane, int xe_col) {
    constexpr int rows[4] = {1, 2, 0, 3};            // own rows y, y+1, then halo rows y-1, y+2
    constexpr int kBytes = E * (int)sizeof(T);
#pragma unroll
    for (int pl = 0; pl < 2; ++pl) {
        int zz = z + pl;
        zz = zz < 0 ? 0 : (zz > nz - 1 ? nz - 1 : zz);
        const T* __restrict__ b = uin + zz * sz;
#pragma unroll
        for (int i = 0; i < 4; ++i) {
            T* dst = slot + (pl * 4 + i) * stride;
            const T* __restrict__ row = b + ro[rows[i]];
            if constexpr (VEC) {
#pragma unroll
                for (int off = 0; off < kBytes; off += 16)
                    s3_cp_async(dst + off / (int)sizeof(T), row + xc[0] + off / (int)sizeof(T), kBytes < 16 ? kBytes : 16);
            } else {
#pragma unroll
                for (int e = 0; e < E; ++e) s3_cp_async(dst + e, row + xc[e], (int)sizeof(T));
            }
        }
        T* ed = eslot + pl * 6;
        if constexpr (SHIFT) {
            if (lane == 0) {                         // xe_col = max(x0 - 2, 0): even, the two columns as one copy
                s3_cp_async(ed + 0, b + ro[1] + xe_col, 2 * (int)sizeof(T));
                s3_cp_async(ed + 2, b + ro[2] + xe_col, 2 * (int)sizeof(T));
                s3_cp_async(ed + 4, b + ro[0] + xe_col + 1, (int)sizeof(T));
                s3_cp_async(ed + 5, b + ro[3] + xe_col + 1, (int)sizeof(T));
            }
        } else {
            if (lane == 0 || lane == 31) {
                s3_cp_async(ed + 1, b + ro[1] + xe_col, (int)sizeof(T));
                s3_cp_async(ed + 3, b + ro[2] + xe_col, (int)sizeof(T));
            }
        }
    }
}
template <typename T, int E>
__device__ __forceinline__ void s3_read_piece(const T* __restrict__ p, T (&v)[E]) {
    constexpr int V = 16 / (int)sizeof(T) < E ? 16 / (int)sizeof(T) : E;       // nodes per shared-memory access
#pragma unroll
    for (int c = 0; c < E / V; ++c) {
        if constexpr (V * sizeof(T) == 16) {
            const typename VecOf<T>::type q = *reinterpret_cast<const typename VecOf<T>::type*>(p + c * V);
            if constexpr (VecOf<T>::V == 4) { v[c * V] = q.x; v[c * V + 1] = q.y; v[c * V + 2] = q.z; v[c * V + 3] = q.w; }
            else { v[c * V] = q.x; v[c * V + 1] = q.y; }
        } else {
            const float2 q = *reinterpret_cast<const float2*>(p + c * V);          // fp32, two nodes per lane
            v[c * V] = q.x; v[c * V + 1] = q.y;
        }
    }
}
template <typename T, int E, bool SHIFT>
__device__ __forceinline__ void s3_read_pair(const T* __restrict__ slot, const T* __restrict__ eslot, int stride,
                                             bool edge_lane, S3Pair<T, E>& p) {
#pragma unroll
    for (int pl = 0; pl < 2; ++pl) {
        s3_read_piece<T, E>(slot + (pl * 4 + 0) * stride, p.own[pl][0]);
        s3_read_piece<T, E>(slot + (pl * 4 + 1) * stride, p.own[pl][1]);
        s3_read_piece<T, E>(slot + (pl * 4 + 2) * stride, p.halo[pl][0]);
        s3_read_piece<T, E>(slot + (pl * 4 + 3) * stride, p.halo[pl][1]);
        if (edge_lane) {
            const T* ed = eslot + pl * 6;
            p.xe[pl][0] = ed[1]; p.xe[pl][1] = ed[3];
            if constexpr (SHIFT) { p.xe2[pl][0] = ed[0]; p.xe2[pl][1] = ed[2]; p.xh[pl][0] = ed[4]; p.xh[pl][1] = ed[5]; }
        }
    }
}

// a lane's piece, 16-byte stores (E * sizeof(T) is a multiple of 16)
template <typename T, int E>
__device__ __forceinline__ void s3_store_piece(T* __restrict__ p, const T (&v)[E]) {
    constexpr int V = VecOf<T>::V;
    static_assert(E % V == 0, "piece of 16-byte vectors");
#pragma unroll
    for (int c = 0; c < E / V; ++c) {
        T t[V];
#pragma unroll
        for (int e = 0; e < V; ++e) t[e] = v[c * V + e];
        st_vec(p + c * V, t);
    }
}

// v[e] <- the value one node to the left: the left lane's v[E-1] at e = 0 (lane 0: `edge`)
template <typename T, int E>
__device__ __forceinline__ void s3_shift(const T (&v)[E], T edge, int lane, T (&out)[E]) {
    T l = __shfl_up_sync(0xffffffffu, v[E - 1], 1);
    if (lane == 0) l = edge;
    out[0] = l;
#pragma unroll
    for (int e = 1; e < E; ++e) out[e] = v[e - 1];
}

// Lanes start at group column 0 of the row (so that a lane's piece is 16-byte aligned in phase 0); group rows and
// plane pairs start at index 1.  Group indices 0 and last of every axis are the shell's: computed here on clamped
// garbage where a lane happens to hold them, never stored.
//
// Phase 1, SHIFTED form (VEC && PH == 1): the groups start at odd columns, so a lane-aligned piece would be
// misaligned by one node and every global access a scalar one (measured: 349 us against 194 us for the aligned
// phase, fp32 512^3).  Instead a lane HOLDS the aligned nodes x0 .. x0+E-1 as in phase 0 and COMPUTES the groups
// of nodes x0-1 .. x0+E-2: its first node comes from the left lane (one shuffle per row kind), its last node goes
// to the right lane's first group, and the new value of node x0-1 travels back to the left lane for the aligned
// store.  Lane 0 takes the incoming values from two extra columns copied with the pair and stores node x0-1
// itself; lane 31 stores all but its last node.
template <typename T, int PH, bool VEC, int NG, int RING>
__global__ void __launch_bounds__(32 * kS3Warps, GE_S3D_MINB)
ge3d_stream_kernel(const T* __restrict__ uin, T* __restrict__ uout, int nx, int ny, int nz,
                   const Coef3<T>* __restrict__ coef, int kseg) {
    constexpr unsigned FULL = 0xffffffffu;
    constexpr int E = 2 * NG;
    constexpr bool SHIFT = VEC && PH == 1;
    const int lane = threadIdx.x;
    const int wx = (int)threadIdx.y % kS3Wx, wy = (int)threadIdx.y / kS3Wx;
    const int x0 = E * (((int)blockIdx.x * kS3Wx + wx) * 32 + lane) - (SHIFT ? 0 : PH);   // first node the lane holds
    const int xg = SHIFT ? x0 - 1 : x0;                                                  // first node of its groups
    // group rows and plane pairs: index PH (the first FULL one) .. ; a row / pair cut by a face is the shell's
    const int y0 = 2 * (PH + (int)blockIdx.y * kS3Wy + wy) - PH;
    if (!(y0 + 1 < ny)) return;                                      // the whole warp: its group row is cut or beyond
    const int kend = PH + (nz - PH) / 2;                             // full pairs: PH .. kend-1
    const int k0 = PH + (int)blockIdx.z * kseg;
    const int k1 = k0 + kseg < kend ? k0 + kseg : kend;
    if (k0 >= k1) return;
    const T r = coef->r, c1 = coef->c1, c2 = coef->c2, c3 = coef->c3;
    // a neighbour one step outside the box is the face's value (ge_level3d.cuh group3d val())
    const T lo0 = coef->lo[0], hi0 = coef->hi[0], lo1 = coef->lo[1], hi1 = coef->hi[1], lo2 = coef->lo[2], hi2 = coef->hi[2];
    const bool ylo = y0 - 1 < 0, yhi = y0 + 2 >= ny;                 // warp-uniform
    const int64_t sy = nx, sz = (int64_t)nx * ny;
    int xc[E];
#pragma unroll
    for (int e = 0; e < E; ++e) { const int x = x0 + e; xc[e] = x < 0 ? 0 : (x > nx - 1 ? nx - 1 : x); }
    if (VEC) xc[0] = x0 > nx - E ? nx - E : x0;                       // nx % E == 0: the piece clamped as a whole
    bool deep[NG + 1];                       // the group is full in x; [NG]: the right lane's first group (shifted form)
#pragma unroll
    for (int g = 0; g <= NG; ++g) deep[g] = xg + 2 * g >= 0 && xg + 2 * g + 1 < nx;
    const bool xlo = xg - 1 < 0, xhi = xg + E >= nx;
    // shifted form: the groups cut by the x faces are computed here as well (cut4_solve of ge_level3d.cuh) -- low:
    // group (-1, 0), the first group of the lane at x0 = 0; high: group (nx-1, nx), computed by the lane that holds
    // node nx-1 from its unshifted values
    const bool cut_lo = SHIFT && x0 == 0, cut_hi = SHIFT && x0 == nx - E;
    const int64_t ro[4] = {(int64_t)(ylo ? 0 : y0 - 1) * sy, (int64_t)y0 * sy, (int64_t)(y0 + 1) * sy,
                           (int64_t)(yhi ? ny - 1 : y0 + 2) * sy};
    const bool edge_lane = SHIFT ? lane == 0 : (lane == 0 || lane == 31);
    int xe_col = SHIFT ? x0 - 2 : (lane == 0 ? x0 - 1 : x0 + E);
    constexpr int kEdgeW = SHIFT ? 2 : 1;                            // the shifted form copies xe_col and xe_col + 1
    xe_col = xe_col < 0 ? 0 : (xe_col > nx - kEdgeW ? nx - kEdgeW : xe_col);

    extern __shared__ __align__(16) unsigned char s3_smem[];
    const int stride = E * 32 * kS3Warps;                            // elements between two pieces of a thread
    constexpr int kSlot = S3Slot<T, E>::elems;                       // elements of one ring slot (all threads)
    T* ring = reinterpret_cast<T*>(s3_smem) + E * ((int)threadIdx.y * 32 + lane);
    T* ering = reinterpret_cast<T*>(s3_smem) + S3Slot<T, E>::pieces + ((int)threadIdx.y * 2 + (lane == 31)) * kS3Edge;

    // pair k0 and the upper plane of the pair below it go through the ring as well (slot 0, then it is free)
    T prevU[2][E];                    // rows y, y+1 of the plane below the pair (shifted form: of the nodes xg ..)
    T prevLast[2];                    // ... of the lane's last node x0+E-1 (shifted form, for the high cut group)
    S3Pair<T, E> cur;
    s3_request_pair<T, E, VEC, SHIFT>(uin, sz, ro, xc, 2 * k0 - PH - 2, nz, ring, ering, stride, lane, xe_col);
    s3_commit();
    s3_wait<0>();
    s3_read_pair<T, E, SHIFT>(ring, ering, stride, edge_lane, cur);
#pragma unroll
    for (int rr = 0; rr < 2; ++rr) {                                 // plane 1 of that "pair" = plane 2 k0 - PH - 1
        if constexpr (SHIFT) s3_shift<T, E>(cur.own[1][rr], cur.xe[1][rr], lane, prevU[rr]);
        else {
#pragma unroll
            for (int e = 0; e < E; ++e) prevU[rr][e] = cur.own[1][rr][e];
        }
        prevLast[rr] = cur.own[1][rr][E - 1];
        if (2 * k0 - PH - 1 < 0) {
#pragma unroll
            for (int e = 0; e < E; ++e) prevU[rr][e] = lo2;
            prevLast[rr] = lo2;
        }
    }
    s3_request_pair<T, E, VEC, SHIFT>(uin, sz, ro, xc, 2 * k0 - PH, nz, ring, ering, stride, lane, xe_col);
    s3_commit();
    s3_wait<0>();
    s3_read_pair<T, E, SHIFT>(ring, ering, stride, edge_lane, cur);
#pragma unroll
    for (int q = 0; q < RING - 1; ++q) {
        s3_request_pair<T, E, VEC, SHIFT>(uin, sz, ro, xc, 2 * (k0 + 1 + q) - PH, nz, ring + q * kSlot, ering + q * kSlot,
                                          stride, lane, xe_col);
        s3_commit();
    }
    int rslot = 0;                    // ring slot of pair k+1

#pragma unroll 1
    for (int k = k0; k < k1; ++k) {
        const int z0 = 2 * k - PH;
        // pair k+RING goes into the slot pair k held (read at the previous iteration); then pair k+1 must have landed
        const int wslot = rslot == 0 ? RING - 1 : rslot - 1;
        s3_request_pair<T, E, VEC, SHIFT>(uin, sz, ro, xc, z0 + 2 * RING, nz, ring + wslot * kSlot, ering + wslot * kSlot,
                                          stride, lane, xe_col);
        s3_commit();
        s3_wait<RING - 1>();
        const T* __restrict__ nslot = ring + rslot * kSlot;
        const T* __restrict__ neslot = ering + rslot * kSlot;
        // the values the groups are computed from, for the nodes xg .. xg+E-1:
        T O[2][2][E], H[2][2][E], NL[2][E];      // pair, rows y-1 / y+2 of its planes, rows y, y+1 of the plane above
        T lf[2][2], rt[2][2];                    // columns xg-1 and xg+E of the pair's four rows
        T nlast[2];                              // rows y, y+1 of the plane above at the lane's last node
        {
            T nlow[2][E];
            s3_read_piece<T, E>(nslot + 0 * stride, nlow[0]);
            s3_read_piece<T, E>(nslot + 1 * stride, nlow[1]);
            nlast[0] = z0 + 2 >= nz ? hi2 : nlow[0][E - 1];
            nlast[1] = z0 + 2 >= nz ? hi2 : nlow[1][E - 1];
            if constexpr (SHIFT) {
                T ne[2] = {T(0), T(0)};
                if (lane == 0) { ne[0] = neslot[1]; ne[1] = neslot[3]; }
#pragma unroll
                for (int rr = 0; rr < 2; ++rr) s3_shift<T, E>(nlow[rr], ne[rr], lane, NL[rr]);
#pragma unroll
                for (int pl = 0; pl < 2; ++pl)
#pragma unroll
                    for (int rr = 0; rr < 2; ++rr) {
                        s3_shift<T, E>(cur.own[pl][rr], cur.xe[pl][rr], lane, O[pl][rr]);
                        s3_shift<T, E>(cur.halo[pl][rr], cur.xh[pl][rr], lane, H[pl][rr]);
                        T l2 = __shfl_up_sync(FULL, cur.own[pl][rr][E - 2], 1);
                        if (lane == 0) l2 = cur.xe2[pl][rr];
                        lf[pl][rr] = l2;
                        rt[pl][rr] = cur.own[pl][rr][E - 1];
                    }
            } else {
#pragma unroll
                for (int pl = 0; pl < 2; ++pl)
#pragma unroll
                    for (int rr = 0; rr < 2; ++rr) {
#pragma unroll
                        for (int e = 0; e < E; ++e) {
                            O[pl][rr][e] = cur.own[pl][rr][e]; H[pl][rr][e] = cur.halo[pl][rr][e];
                            if (pl == 0) NL[rr][e] = nlow[rr][e];
                        }
                        lf[pl][rr] = __shfl_up_sync(FULL, cur.own[pl][rr][E - 1], 1);
                        rt[pl][rr] = __shfl_down_sync(FULL, cur.own[pl][rr][0], 1);
                        if (lane == 0) lf[pl][rr] = cur.xe[pl][rr];
                        if (lane == 31) rt[pl][rr] = cur.xe[pl][rr];
                    }
            }
        }
        // neighbours outside the box
#pragma unroll
        for (int pl = 0; pl < 2; ++pl)
#pragma unroll
            for (int rr = 0; rr < 2; ++rr) {
                if (xlo) lf[pl][rr] = lo0;
                if (xhi) rt[pl][rr] = hi0;
#pragma unroll
                for (int e = 0; e < E; ++e) {
                    if (!VEC && xg + e >= nx) O[pl][rr][e] = hi0;    // (VEC: a lane is inside or outside as a whole)
                    if (rr == 0 && ylo) H[pl][0][e] = lo1;
                    if (rr == 1 && yhi) H[pl][1][e] = hi1;
                    if (pl == 0 && z0 + 2 >= nz) NL[rr][e] = hi2;
                }
            }
        T nw[2][2][E];                // new values of the nodes xg .. xg+E-1: [plane][row][node]
#pragma unroll
        for (int g = 0; g < NG; ++g) {
            // right-hand sides, member d = dx + 2 dy + 4 dz (ge_level3d.cuh group3d)
            T R[8];
#pragma unroll
            for (int d = 0; d < 8; ++d) {
                const int dx = d & 1, dy = (d >> 1) & 1, dz = (d >> 2) & 1;
                const T o = O[dz][dy][2 * g + dx];
                const T ox = dx ? (g + 1 < NG ? O[dz][dy][g + 1 < NG ? 2 * g + 2 : 0] : rt[dz][dy])
                                : (g > 0 ? O[dz][dy][g > 0 ? 2 * g - 1 : 0] : lf[dz][dy]);
                const T oy = H[dz][dy][2 * g + dx];
                const T oz = dz ? NL[dy][2 * g + dx] : prevU[dy][2 * g + dx];
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
#pragma unroll
            for (int d = 0; d < 8; ++d) nw[(d >> 2) & 1][(d >> 1) & 1][2 * g + (d & 1)] = R[d] - W[d];
            if constexpr (SHIFT) {
                if (g == 0 && cut_lo) {              // group (-1, 0): its members dx = 1 are node 0
                    T R4[4], x4[4];
#pragma unroll
                    for (int j = 0; j < 4; ++j) R4[j] = R[1 + 2 * j];
                    cut4_solve<T>(R4, r, lo0, coef->q1, coef->q2, coef->q3, x4);
#pragma unroll
                    for (int j = 0; j < 4; ++j) nw[j >> 1][j & 1][1] = x4[j];
                }
            }
        }
        T hi_new[4] = {T(0), T(0), T(0), T(0)};      // new values of node nx-1, j = dy + 2 dz (shifted form, cut_hi)
        if constexpr (SHIFT) {
            if (cut_hi) {                            // group (nx-1, nx): its members dx = 0 are node nx-1 = the lane's last
                T R4[4];
#pragma unroll
                for (int j = 0; j < 4; ++j) {
                    const int dy = j & 1, dz = j >> 1;
                    const T o = cur.own[dz][dy][E - 1], ox = cur.own[dz][dy][E - 2];
                    const T oy = dy ? (yhi ? hi1 : cur.halo[dz][1][E - 1]) : (ylo ? lo1 : cur.halo[dz][0][E - 1]);
                    const T oz = dz ? nlast[dy] : prevLast[dy];
                    R4[j] = fma(r, ((ox - o) + (oy - o)) + (oz - o), o);
                }
                cut4_solve<T>(R4, r, hi0, coef->q1, coef->q2, coef->q3, hi_new);
            }
        }
        T* __restrict__ ob = uout + (int64_t)z0 * sz + ro[1] + x0;   // the lane's aligned piece (VEC)
        if constexpr (SHIFT) {
            // out[e] = node x0 + e = nw[e + 1]; the last one is the right lane's nw[0] (the next warp's lane 0 stores
            // it itself), or the high cut group's
            const bool in_row = x0 <= nx - E;
            const bool has_last = cut_hi || (lane != 31 && x0 < nx - E);
#pragma unroll
            for (int dz = 0; dz < 2; ++dz)
#pragma unroll
                for (int dy = 0; dy < 2; ++dy) {
                    T out[E];
#pragma unroll
                    for (int e = 0; e + 1 < E; ++e) out[e] = nw[dz][dy][e + 1];
                    out[E - 1] = __shfl_down_sync(FULL, nw[dz][dy][0], 1);
                    if (cut_hi) out[E - 1] = hi_new[dy + 2 * dz];
                    T* __restrict__ o2 = ob + dz * sz + dy * sy;
                    if (in_row) {
                        if (has_last) {
                            s3_store_piece<T, E>(o2, out);
                        } else {
#pragma unroll
                            for (int e = 0; e + 1 < E; ++e) o2[e] = out[e];
                        }
                        if (lane == 0 && x0 > 0) o2[-1] = nw[dz][dy][0];
                    }
                }
        } else {
            bool all = VEC, stored = false;
#pragma unroll
            for (int g = 0; g < NG; ++g) all = all && deep[g];
            if constexpr (E * sizeof(T) == 16) {
                if (all) {
#pragma unroll
                    for (int dz = 0; dz < 2; ++dz)
#pragma unroll
                        for (int dy = 0; dy < 2; ++dy) st_vec(ob + dz * sz + dy * sy, nw[dz][dy]);
                    stored = true;
                }
            }
            if (!stored) {
#pragma unroll
                for (int g = 0; g < NG; ++g)
                    if (deep[g]) {
#pragma unroll
                        for (int dz = 0; dz < 2; ++dz)
#pragma unroll
                            for (int dy = 0; dy < 2; ++dy) {
                                T* __restrict__ o2 = ob + dz * sz + dy * sy + 2 * g;
                                if constexpr (VEC) {
                                    typename Vec2<T>::type q; q.x = nw[dz][dy][2 * g]; q.y = nw[dz][dy][2 * g + 1];
                                    *reinterpret_cast<typename Vec2<T>::type*>(o2) = q;
                                } else { o2[0] = nw[dz][dy][2 * g]; o2[1] = nw[dz][dy][2 * g + 1]; }
                            }
                    }
            }
        }
        // slide up by one pair: the upper plane becomes the plane below, pair k+1 comes out of its ring slot
#pragma unroll
        for (int rr = 0; rr < 2; ++rr) {
#pragma unroll
            for (int e = 0; e < E; ++e) prevU[rr][e] = O[1][rr][e];
            prevLast[rr] = cur.own[1][rr][E - 1];
        }
        s3_read_pair<T, E, SHIFT>(nslot, neslot, stride, edge_lane, cur);
        rslot = rslot + 1 == RING ? 0 : rslot + 1;
    }
}

// The groups cut by a face.  `faces`: 3 bits per blockIdx.z = face (axis * 2 + side) with cut groups;
// the face's two other axes are tiled by the block; group3d does faces, edges and corners (by elimination).
// Groups on an edge or corner of the box belong to two or three faces and are written by each with the same value.
template <typename T, int PH>
__global__ void __launch_bounds__(128)
ge3d_shell_kernel(const T* __restrict__ uin, T* __restrict__ uout, int nx, int ny, int nz,
                  const Coef3<T>* __restrict__ coef, unsigned faces) {
    const Coef3<T> k = *coef;
    const int n[3] = {nx, ny, nz};
    const int face = (faces >> (3 * blockIdx.z)) & 7, ax = face >> 1, side = face & 1;
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
    constexpr int NG = S3Cfg<T>::ng, RING = S3Cfg<T>::ring;
    constexpr size_t smem = (size_t)RING * S3Slot<T, 2 * NG>::elems * sizeof(T);
    if (smem > 48 * 1024) {                    // idempotent, a few microseconds against a level of >= 100
        const cudaError_t e = cudaFuncSetAttribute(ge3d_stream_kernel<T, PH, VEC, NG, RING>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
        if (e != cudaSuccess) return e;
    }
    ge3d_stream_kernel<T, PH, VEC, NG, RING><<<grid, dim3(32, kS3Warps), smem, s>>>(uin, uout, nx, ny, nz, coef, kseg);
    return cudaGetLastError();
}

// aux / ev_in / ev_out (optional): the shell kernel runs on the stream `aux`, beside the streaming kernel -- both
// read the old level and write disjoint parts of the new one; ev_in orders it after the work already on `s`,
// ev_out makes `s` wait for it.
template <typename T>
inline cudaError_t stream3d_launch(const T* uin, T* uout, int64_t nx, int64_t ny, int64_t nz, const Coef3<T>* coef,
                                   int phase, int sm_count, cudaStream_t s, int* launches, cudaStream_t aux = nullptr,
                                   cudaEvent_t ev_in = nullptr, cudaEvent_t ev_out = nullptr) {
    *launches = 0;
    auto last = [&](int64_t n) { return (n - 1 + phase) / 2; };         // group index of the last anchor <= n-1
    // full groups (both nodes in the box) per axis: indices phase .. phase + g - 1; the streaming kernel's
    const int64_t gx = (nx - phase) / 2, gy = (ny - phase) / 2, gz = (nz - phase) / 2;
    // faces with cut groups (anchor -1, or anchor n-1): the shell kernel's
    unsigned faces = 0; int nfaces = 0;
    const int64_t nn[3] = {nx, ny, nz};
    constexpr int kE = 2 * S3Cfg<T>::ng;
    const bool vec = nx % kE == 0 && (((uintptr_t)uin | (uintptr_t)uout) % (kE * sizeof(T))) == 0;
    const bool have_main = gx > 0 && gy > 0 && gz > 0;
    // the shifted form (vec, phase 1) computes the groups cut by the x faces itself; those cut by another face
    // as well are on that face's list
    const bool x_in_main = have_main && vec && phase == 1;
    for (int a = 0; a < 3; ++a) {
        if (a == 0 && x_in_main) continue;
        if (phase == 1) { faces |= (unsigned)(2 * a) << (3 * nfaces); ++nfaces; }
        if (2 * last(nn[a]) - phase + 1 >= nn[a]) { faces |= (unsigned)(2 * a + 1) << (3 * nfaces); ++nfaces; }
    }
    auto groups = [&](int64_t n) { return last(n) + 1; };
    const int64_t ax = groups(nx), ay = groups(ny), az = groups(nz);
    const int64_t gmax = ax > ay ? (ax > az ? ax : az) : (ay > az ? ay : az);
    // The shell kernel is small and latency-bound; it runs beside the streaming kernel on another stream (both read the
    // old level and write disjoint parts of the new one).  GE_S3D_MODE 0: shell first on `aux`, the streaming kernel
    // on `s` fills the rest of the chip; 1: the streaming kernel first on `s`, the shell after it on `aux`; 2: the
    // streaming kernel on `aux` (a high-priority stream: its CTAs go first), the shell on `s`.
    const bool side = aux && ev_in && ev_out && nfaces > 0;
    constexpr int kMode = GE_S3D_MODE;
    cudaStream_t s_shell = side ? (kMode == 2 ? s : aux) : s;
    cudaStream_t s_main = side && kMode == 2 ? aux : s;
    auto launch_shell = [&]() -> cudaError_t {
        if (nfaces == 0) return cudaSuccess;
        dim3 sblock(32, 4), sgrid((unsigned)((gmax + 31) / 32), (unsigned)((gmax + 3) / 4), (unsigned)nfaces);
#ifndef GE_S3D_NOSHELL          // (timing diagnostic only: without the shell launch the cut groups are not computed)
        if (phase == 0) ge3d_shell_kernel<T, 0><<<sgrid, sblock, 0, s_shell>>>(uin, uout, (int)nx, (int)ny, (int)nz, coef, faces);
        else            ge3d_shell_kernel<T, 1><<<sgrid, sblock, 0, s_shell>>>(uin, uout, (int)nx, (int)ny, (int)nz, coef, faces);
#endif
        *launches += 1;
        return cudaGetLastError();
    };
    auto launch_main = [&]() -> cudaError_t {
        if (!have_main) return cudaSuccess;
        // z segments: enough CTAs for ~8 resident CTAs on every SM, at least 8 pairs per segment
        // lanes start at group column 0 and hold NG group columns each; the last deep group column is index gx
        const int64_t per_cta = 32 * kS3Wx * S3Cfg<T>::ng;
        const int64_t bx = (gx + phase + per_cta - 1) / per_cta;
        const int64_t ctas_xy = bx * ((gy + kS3Wy - 1) / kS3Wy);
#ifdef GE_S3D_SEGS                // (sweep knob: a fixed number of z segments; 7 .. 23 measured within 1 %)
        int64_t segs = GE_S3D_SEGS;
#else
        int64_t segs = (8 * (int64_t)sm_count + ctas_xy - 1) / ctas_xy;
#endif
        if (segs > gz / 8) segs = gz / 8;
        if (segs < 1) segs = 1;
        const int kseg = (int)((gz + segs - 1) / segs);
        dim3 grid((unsigned)bx, (unsigned)((gy + kS3Wy - 1) / kS3Wy), (unsigned)((gz + kseg - 1) / kseg));
        *launches += 1;
        if (phase == 0) return vec ? stream3d_launch_one<T, 0, true>(uin, uout, (int)nx, (int)ny, (int)nz, coef, kseg, grid, s_main)
                                   : stream3d_launch_one<T, 0, false>(uin, uout, (int)nx, (int)ny, (int)nz, coef, kseg, grid, s_main);
        return vec ? stream3d_launch_one<T, 1, true>(uin, uout, (int)nx, (int)ny, (int)nz, coef, kseg, grid, s_main)
                   : stream3d_launch_one<T, 1, false>(uin, uout, (int)nx, (int)ny, (int)nz, coef, kseg, grid, s_main);
    };
    cudaError_t e = cudaSuccess;
    if (side) {
        e = cudaEventRecord(ev_in, s);
        if (e == cudaSuccess) e = cudaStreamWaitEvent(aux, ev_in, 0);
        if (e != cudaSuccess) return e;
    }
    if (kMode == 0) {
        e = launch_shell();
        if (e == cudaSuccess) e = launch_main();
    } else {
        e = launch_main();
        if (e == cudaSuccess) e = launch_shell();
    }
    if (e != cudaSuccess) return e;
    if (side) {
        e = cudaEventRecord(ev_out, aux);
        if (e == cudaSuccess) e = cudaStreamWaitEvent(s, ev_out, 0);
    }
    return e;
}

}  // namespace ge
