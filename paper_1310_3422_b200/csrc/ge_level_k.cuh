// ge_level_k.cuh -- strategy A for the paper's general scheme, sub-domain length
// k >= 2 (the paper's own runs use k = 16):
// one kernel launch per level, one HBM round trip per level.
//
// Rule table.  Class of node i: c = (i - phase*k) mod 2k.
//   c = 0      right member of the confluence pair (i-1, i)      Eq (4)
//   c = 1..k-1 Saul'yev A, ascending i, uses new_{i-1}           Eq (1)
//   c = k..2k-2 Saul'yev B, descending i, uses new_{i+1}         Eq (2)
//   c = 2k-1   left member of the pair (i, i+1)                  Eq (3)
// A pair with a boundary member gives its interior member Eq (1)/(2) with the
// boundary value as new-level neighbour; sweeps that reach a boundary read it.
//
// Ownership is the paper's: a thread owns one UNIT = 2k
// consecutive nodes c = 0 .. 2k-1 (the paper's "sub-domain couple" seen from its
// left wall): it forms the right member of the pair at its left wall, sweeps A
// k-1 nodes to the right, forms the left member of the pair at its right wall and
// sweeps B k-1 nodes to the left -- two independent serial chains, everything
// it reads beyond its own nodes are the two old values either side.  What is not
// the paper's: threads share only OLD values (one barrier after every thread has
// read its four, then the unit is updated in place), the CTA stages its units through shared memory so
// that HBM sees coalesced 128-byte lines (a unit is padded to 2k+1 words, which
// makes the strided per-thread accesses bank-conflict-free), and the arithmetic
// is the "value + correction" form of ge_common.cuh:
//   Eq (1): new_i = old_i + e ((new_{i-1} - old_i) + (old_{i+1} - old_i)),  e = r/(1+r)
//   Eq (2): new_i = old_i + e ((new_{i+1} - old_i) + (old_{i-1} - old_i))
//   pair  : pair_update (Eqs (3),(4) factored)
#pragma once
#include "ge_common.cuh"

namespace ge {

constexpr int kLevelKThreads = 128;

struct LevelKGeom {
    int k;
    int phase;
    int upc;               // units per CTA (<= kLevelKThreads)
    int64_t s0;            // node where unit 0 starts: 0 (phase 0) or -k (phase 1)
    int64_t units;         // units per rod
};

inline LevelKGeom level_k_geom(int k, int phase, int64_t nx, size_t elem, size_t smem_budget) {
    LevelKGeom g;
    g.k = k; g.phase = phase;
    g.s0 = phase ? -(int64_t)k : 0;
    g.units = (nx - g.s0) / (2 * (int64_t)k) + 1;          // all units with start <= N
    int64_t upc = (int64_t)((smem_budget - 4 * elem) / ((size_t)(2 * k + 1) * elem));
    if (upc > kLevelKThreads) upc = kLevelKThreads;
    if (upc > g.units) upc = g.units;
    g.upc = (int)upc;                                       // 0: k too large for shared memory
    return g;
}
inline size_t level_k_smem(const LevelKGeom& g, size_t elem) {
    return ((size_t)g.upc * (2 * g.k + 1) + 4) * elem;
}

template <typename T>
__global__ void __launch_bounds__(kLevelKThreads)
ge1d_level_k_kernel(const T* __restrict__ uin, T* __restrict__ uout, int64_t nx, int64_t batch,
                    const Coef1<T>* __restrict__ coef, const LevelKGeom g) {
    extern __shared__ __align__(16) unsigned char levelk_smem[];
    const int k = g.k, two_k = 2 * g.k, pitch = 2 * g.k + 1;
    const int span = g.upc * two_k;                        // nodes of this CTA's units
    T* so = reinterpret_cast<T*>(levelk_smem);             // unit u at u*pitch; old values, then new in place
    T* sh = so + (size_t)g.upc * pitch;                    // old values of nodes S-2, S-1, S+span, S+span+1
    const int64_t S = g.s0 + (int64_t)blockIdx.x * span;   // first node of the CTA
    const int64_t N = nx;
    for (int64_t rod = blockIdx.y; rod < batch; rod += gridDim.y) {
        const Coef1<T> c = coef[rod];
        const T* __restrict__ in = uin + rod * nx;
        T* __restrict__ out = uout + rod * nx;
        auto node_value = [&](int64_t i) -> T {            // old value of node i, boundaries included
            if (i < 0 || i > N + 1) return T(0);
            if (i == 0) return c.lo;
            if (i == N + 1) return c.hi;
            return __ldg(in + (i - 1));
        };
        // ---- coalesced load into the padded layout: one cp.async per node (HBM -> shared memory without
        //      a register in between, all of a thread's copies in flight together) ----
        {
            int q = threadIdx.x / two_k, rem = threadIdx.x % two_k;
            const int dq = kLevelKThreads / two_k, dr = kLevelKThreads % two_k;
            for (int j = threadIdx.x; j < span; j += kLevelKThreads) {
                const int64_t i = S + j;
                T* dst = so + q * pitch + rem;
                if (i >= 1 && i <= N) {
                    const uint32_t d32 = (uint32_t)__cvta_generic_to_shared(dst);
                    if constexpr (sizeof(T) == 8)
                        asm volatile("cp.async.ca.shared.global [%0], [%1], 8;" ::"r"(d32), "l"(in + (i - 1)) : "memory");
                    else
                        asm volatile("cp.async.ca.shared.global [%0], [%1], 4;" ::"r"(d32), "l"(in + (i - 1)) : "memory");
                } else {
                    *dst = node_value(i);
                }
                q += dq; rem += dr;
                if (rem >= two_k) { rem -= two_k; ++q; }
            }
            if (threadIdx.x < 4) {
                const int64_t i = threadIdx.x < 2 ? S - 2 + threadIdx.x : S + span + (threadIdx.x - 2);
                sh[threadIdx.x] = node_value(i);
            }
            asm volatile("cp.async.wait_all;" ::: "memory");
        }
        __syncthreads();
        // ---- one unit per thread, in place ----
        const int t = threadIdx.x;
        const int64_t s = S + (int64_t)t * two_k;          // node with c = 0
        const bool mine = t < g.upc && s <= N;
        T* o = so + t * pitch;
        T om2 = T(0), om1 = T(0), op0 = T(0), op1 = T(0);  // old values just outside the unit
        if (mine) {
            om2 = t > 0 ? o[-pitch + two_k - 2] : sh[0];
            om1 = t > 0 ? o[-pitch + two_k - 1] : sh[1];
            op0 = t + 1 < g.upc ? o[pitch] : sh[2];
            op1 = t + 1 < g.upc ? o[pitch + 1] : sh[3];
        }
        __syncthreads();                                   // neighbours have read my edge values: overwrite freely
        if (mine) {
            const int64_t e = s + two_k - 1;               // node with c = 2k-1
            // (1) right member of the pair (s-1, s), (3) left member of the pair (e, e+1)
            T prev = c.lo;                                 // new value of the node left of the A sweep
            T next = c.hi;                                 // new value of the node right of the B sweep
            const T o0 = o[0], o1 = o[1], oe1 = o[two_k - 2], oe = o[two_k - 1];
            if (s >= 1) {
                T lo_, hi_;
                pair_update_bc(om2, om1, o0, o1, c, s - 1 == 0, false, lo_, hi_);
                prev = hi_;
            }
            if (e >= 1 && e <= N) {
                T lo_, hi_;
                pair_update_bc(oe1, oe, op0, op1, c, false, e + 1 == N + 1, lo_, hi_);
                next = lo_;
            }
            // (2) Saul'yev A ascending from the left wall and (4) Saul'yev B descending from the right
            // wall, one node of each per iteration: two independent chains that meet in the middle.
            // Every iteration reads its four old values before it writes, so the update is in place.
            T a_old = o1;                                  // old value of the A node of this iteration
            T b_old = oe1;                                 // old value of the B node of this iteration
            o[0] = prev; o[two_k - 1] = next;
#pragma unroll 4
            for (int m = 1; m < k; ++m) {
                const int ja = m, jb = two_k - 1 - m;
                const T a_nxt = o[ja + 1];                 // old_{i+1} of the A node (jb when the chains meet)
                const T b_nxt = o[jb - 1];                 // old_{i-1} of the B node
                const int64_t ia = s + ja, ib = s + jb;
                if (ia >= 1 && ia <= N) {
                    prev = fma(c.e, (prev - a_old) + (a_nxt - a_old), a_old);
                    o[ja] = prev;
                }
                if (ib >= 1 && ib <= N) {
                    next = fma(c.e, (next - b_old) + (b_nxt - b_old), b_old);
                    o[jb] = next;
                }
                a_old = a_nxt; b_old = b_nxt;
            }
        }
        __syncthreads();
        // ---- coalesced store of the interior nodes ----
        {
            int q = threadIdx.x / two_k, rem = threadIdx.x % two_k;
            const int dq = kLevelKThreads / two_k, dr = kLevelKThreads % two_k;
            for (int j = threadIdx.x; j < span; j += kLevelKThreads) {
                const int64_t i = S + j;
                if (i >= 1 && i <= N) out[i - 1] = so[q * pitch + rem];
                q += dq; rem += dr;
                if (rem >= two_k) { rem -= two_k; ++q; }
            }
        }
        __syncthreads();                                   // the buffers are reused by the next rod
    }
}

}  // namespace ge

// ------------------------------------------------------------------------------------------------
// Strategy C for k >= 2: the whole run of a rod in ONE launch, the rod resident in shared memory
// (the paper's own run shape -- 8208 nodes, sub-domain couples of 32, <= 1200 levels, PAPER.md:204-218
// -- is launch-bound at one launch per level: 6 us per level for 0.1 us of work).
// One CTA per rod, one thread per unit as above; per level every thread reads the two old values either
// side of its unit, the CTA synchronises, the unit is updated in place, the CTA synchronises -- the
// paper's two barriers per level PAIR become two per level, but they are CTA barriers that cost ~50 ns
// and there is no block-to-block ordering left to luck.  The unit decomposition shifts by
// k nodes between levels, so the layout is linear in the node index, skewed by one word per 32 (node i
// at i + i/32): threads 2k nodes apart fall into different banks whatever the phase.
namespace ge {

struct RodKGeom {
    int k;
    int threads;           // >= units of either phase, multiple of 32, <= 1024
    size_t smem;           // bytes
};
inline RodKGeom rod_k_geom(int k, int64_t nx, size_t elem) {
    RodKGeom g;
    g.k = k;
    const int64_t units = (nx + k) / (2 * (int64_t)k) + 1;            // phase 1 has the most
    g.threads = units <= 1024 ? (int)((units + 31) / 32 * 32) : 0;
    const int64_t words = (nx + 2) + (nx + 2) / 32 + 1;
    g.smem = (size_t)words * elem;
    return g;
}

template <typename T>
__global__ void __launch_bounds__(1024)
ge1d_rod_k_resident_kernel(T* u, int64_t nx, int64_t batch, const Coef1<T>* __restrict__ coef, int k,
                           int phase0, int64_t steps) {
    extern __shared__ __align__(16) unsigned char rodk_smem[];
    T* sm = reinterpret_cast<T*>(rodk_smem);
    const int N = (int)nx, two_k = 2 * k;
    auto at = [&](int i) -> T& { return sm[i + (i >> 5)]; };           // node i, 0 <= i <= N+1
    auto rd = [&](int i) -> T { return (i >= 0 && i <= N + 1) ? sm[i + (i >> 5)] : T(0); };
    const int t = threadIdx.x;
    for (int64_t rod = blockIdx.x; rod < batch; rod += gridDim.x) {
        const Coef1<T> c = coef[rod];
        T* row = u + rod * nx;
        for (int i = t; i <= N + 1; i += blockDim.x) at(i) = i == 0 ? c.lo : (i == N + 1 ? c.hi : row[i - 1]);
        __syncthreads();
#pragma unroll 1
        for (int64_t lev = 0; lev < steps; ++lev) {
            const int phase = (int)((phase0 + lev) & 1);
            const int s = (phase ? -k : 0) + t * two_k;               // node with c = 0
            const int e = s + two_k - 1;                               // node with c = 2k-1
            const bool mine = s <= N;
            T om2 = T(0), om1 = T(0), op0 = T(0), op1 = T(0), o0 = T(0), o1 = T(0), oe1 = T(0), oe = T(0);
            if (mine) {
                om2 = rd(s - 2); om1 = rd(s - 1); o0 = rd(s); o1 = rd(s + 1);
                oe1 = rd(e - 1); oe = rd(e); op0 = rd(e + 1); op1 = rd(e + 2);
            }
            __syncthreads();                                           // everybody has its old wall values
            if (mine) {
                T prev = c.lo, next = c.hi;
                if (s >= 1) {
                    T lo_, hi_;
                    pair_update_bc(om2, om1, o0, o1, c, s - 1 == 0, false, lo_, hi_);
                    prev = hi_;
                    at(s) = prev;
                }
                if (e >= 1 && e <= N) {
                    T lo_, hi_;
                    pair_update_bc(oe1, oe, op0, op1, c, false, e + 1 == N + 1, lo_, hi_);
                    next = lo_;
                    at(e) = next;
                }
                T a_old = o1, b_old = oe1;
#pragma unroll 4
                for (int m = 1; m < k; ++m) {
                    const int ia = s + m, ib = e - m;
                    const T a_nxt = rd(ia + 1);
                    const T b_nxt = rd(ib - 1);
                    if (ia >= 1 && ia <= N) {
                        prev = fma(c.e, (prev - a_old) + (a_nxt - a_old), a_old);
                        at(ia) = prev;
                    }
                    if (ib >= 1 && ib <= N) {
                        next = fma(c.e, (next - b_old) + (b_nxt - b_old), b_old);
                        at(ib) = next;
                    }
                    a_old = a_nxt; b_old = b_nxt;
                }
            }
            __syncthreads();
        }
        for (int i = t; i < N; i += blockDim.x) row[i] = at(i + 1);
        __syncthreads();
    }
}

}  // namespace ge

// ------------------------------------------------------------------------------------------------
// Strategy B for k >= 2: `levels` <= tb levels per HBM round trip on a long rod (the
// paper's own k = 16, on rods that do not fit one CTA).  A CTA owns a tile of `valid` nodes,
// loads them with `halo` more per side into shared memory (the skewed layout of the resident kernel) and
// marches the window through the levels exactly as ge1d_rod_k_resident_kernel marches a rod -- one thread
// per unit of 2k nodes, two CTA barriers per level -- treating whatever lies beyond a cut end as unknown.
// What a cut end spoils: a node of an A sweep is only as good as its unit's left wall pair, a node of a B
// sweep as good as everything from its left neighbour to the right wall pair (neighbours share
// nothing but wall nodes), so the first good node moves inward by at most k+1 nodes per level (the A half
// of the unit the front is in; the unit grid then shifts by k); a unit cut by the window's end is not marched
// at all, which costs one more unit once: halo = tb (k+1) + 2k + 2 nodes.  A window end that IS the rod's end
// holds the Dirichlet node and is exact.  Same expressions as the per-level kernel on the
// same operands: bit-identical.
namespace ge {

struct TemporalKGeom {
    int k, tb;
    int halo;              // nodes per cut side
    int valid;             // nodes a tile delivers
    int window;            // valid + 2 halo
    int threads;           // >= units of a window in either phase (+1 for a straddling unit), multiple of 32
    int64_t tiles;
    size_t smem;
    int64_t end_len;       // > 0: two CTAs per rod that recompute its first / last end_len nodes only (ge_unit_k.cuh)
};
inline TemporalKGeom temporal_k_geom(int k, int tb, int64_t nx, size_t elem, size_t smem_budget) {
    TemporalKGeom g;
    g.k = k; g.tb = tb; g.end_len = 0;
    g.halo = tb * (k + 1) + 2 * k + 2;
    int64_t window = (int64_t)(smem_budget / elem) * 32 / 33 - 8;       // skew: one extra word per 32
    if (window > 1020 * 2 * (int64_t)k) window = 1020 * 2 * (int64_t)k; // <= 1024 threads (units + 2, rounded to warps)
    int64_t valid = window - 2 * g.halo;
    if (valid > nx) valid = nx;
    valid -= valid % 2;
    if (valid < 2 * (int64_t)k || valid < g.halo) { g.valid = 0; g.window = 0; g.threads = 0; g.tiles = 0; g.smem = 0; return g; }
    g.valid = (int)valid;
    g.window = g.valid + 2 * g.halo;
    const int units = g.window / (2 * k) + 2;
    g.threads = (units + 31) / 32 * 32;
    g.tiles = (nx + g.valid - 1) / g.valid;
    const int64_t words = (int64_t)g.window + 4 + (g.window + 4) / 32 + 1;
    g.smem = (size_t)words * elem;
    if (g.threads > 1024) { g.valid = 0; g.tiles = 0; }
    return g;
}
// the same kernel on the two ends of the rod only: windows of end_len + halo nodes
inline TemporalKGeom temporal_k_ends_geom(int k, int tb, int64_t end_len, size_t elem) {
    TemporalKGeom g;
    g.k = k; g.tb = tb; g.end_len = end_len;
    g.halo = tb * (k + 1) + 2 * k + 2;
    g.valid = (int)end_len;
    g.window = g.valid + g.halo;                       // one side of an end window is the rod's end
    g.threads = (g.window / (2 * k) + 2 + 31) / 32 * 32;
    g.tiles = 2;
    g.smem = (size_t)((int64_t)g.window + 4 + (g.window + 4) / 32 + 1) * elem;
    if (g.threads > 1024) { g.valid = 0; g.tiles = 0; }
    return g;
}

template <typename T>
__global__ void __launch_bounds__(1024)
ge1d_temporal_k_kernel(const T* __restrict__ uin, T* __restrict__ uout, int64_t nx, int64_t batch,
                       const Coef1<T>* __restrict__ coef, const TemporalKGeom g, int phase0, int levels) {
    extern __shared__ __align__(16) unsigned char tk_smem[];
    T* sm = reinterpret_cast<T*>(tk_smem);
    const int k = g.k, two_k = 2 * g.k;
    const int64_t N = nx;
    const int t = threadIdx.x;
    // nodes of this tile: valid [v0, v1), window [w0, w1) clipped to the rod with its Dirichlet nodes 0 and N+1
    const int64_t v0 = g.end_len > 0 ? (blockIdx.x == 0 ? 1 : (N + 1 - g.end_len > 1 ? N + 1 - g.end_len : 1))
                                     : 1 + (int64_t)blockIdx.x * g.valid;
    const int64_t v1 = g.end_len > 0 ? (blockIdx.x == 0 ? (1 + g.end_len < N + 1 ? 1 + g.end_len : N + 1) : N + 1)
                                     : (v0 + g.valid < N + 1 ? v0 + g.valid : N + 1);
    const int64_t w0 = v0 - g.halo > 0 ? v0 - g.halo : 0;
    const int64_t w1 = v1 + g.halo < N + 2 ? v1 + g.halo : N + 2;
    const int len = (int)(w1 - w0);
    auto at = [&](int j) -> T& { return sm[j + (j >> 5)]; };                         // window element j = node w0 + j
    auto rd = [&](int j) -> T { return (j >= 0 && j < len) ? sm[j + (j >> 5)] : T(0); };
    for (int64_t rod = blockIdx.y; rod < batch; rod += gridDim.y) {
        const Coef1<T> c = coef[rod];
        const T* __restrict__ in = uin + rod * nx;
        T* __restrict__ out = uout + rod * nx;
        // one cp.async per node: all of a thread's copies are in flight together (a plain load-store loop pays
        // one HBM latency per trip: 30 trips ~ 30 us against ~1 us of levels)
        for (int j = t; j < len; j += blockDim.x) {
            const int64_t i = w0 + j;
            if (i >= 1 && i <= N) {
                const uint32_t d32 = (uint32_t)__cvta_generic_to_shared(&at(j));
                if constexpr (sizeof(T) == 8)
                    asm volatile("cp.async.ca.shared.global [%0], [%1], 8;" ::"r"(d32), "l"(in + (i - 1)) : "memory");
                else
                    asm volatile("cp.async.ca.shared.global [%0], [%1], 4;" ::"r"(d32), "l"(in + (i - 1)) : "memory");
            } else {
                at(j) = i == 0 ? c.lo : c.hi;
            }
        }
        asm volatile("cp.async.wait_all;" ::: "memory");
        __syncthreads();
        // this thread's unit in either phase (window coordinates of its node with c = 0), hoisted out of the level
        // loop; a unit is marched when it lies inside the window together with the two old values either side of
        // it, or when it touches an end of the ROD (then the index-tested path below handles what is missing).
        // A unit cut by an end of the WINDOW is left alone: its nodes are halo that is stale anyway.
        int s_ph[2]; bool run_ph[2], fast_ph[2];
#pragma unroll
        for (int ph = 0; ph < 2; ++ph) {
            const int64_t off = ph ? -(int64_t)k : 0;
            const int64_t sg = off + ((w0 - off) / two_k + t) * two_k;     // w0 - off >= 0
            const int64_t eg = sg + two_k - 1;
            const int s = (int)(sg - w0);
            s_ph[ph] = s;
            const bool inside = s >= 2 && s + two_k + 1 < len;             // nodes s-2 .. e+2 in the window
            fast_ph[ph] = inside && sg >= 2 && eg + 1 <= N;                // ... and all of them interior nodes
            const bool rod_end = (sg < 2 && w0 == 0) || (eg + 1 > N && w1 == N + 2);
            run_ph[ph] = sg <= N && s < len && (inside || rod_end);
        }
#pragma unroll 1
        for (int lev = 0; lev < levels; ++lev) {
            const int phase = (phase0 + lev) & 1;
            const int s = phase ? s_ph[1] : s_ph[0], e = s + two_k - 1;     // window coordinates
            const int64_t sg = w0 + s;                                     // node with c = 0 of this thread's unit
            const bool mine = phase ? run_ph[1] : run_ph[0], fast = phase ? fast_ph[1] : fast_ph[0];
            T om2 = T(0), om1 = T(0), op0 = T(0), op1 = T(0), o0 = T(0), o1 = T(0), oe1 = T(0), oe = T(0);
            if (fast) {
                om2 = at(s - 2); om1 = at(s - 1); o0 = at(s); o1 = at(s + 1);
                oe1 = at(e - 1); oe = at(e); op0 = at(e + 1); op1 = at(e + 2);
            } else if (mine) {
                om2 = rd(s - 2); om1 = rd(s - 1); o0 = rd(s); o1 = rd(s + 1);
                oe1 = rd(e - 1); oe = rd(e); op0 = rd(e + 1); op1 = rd(e + 2);
            }
            __syncthreads();                                           // everybody has its old wall values
            if (fast) {
                // no index tests; the address of a node written is the address it was read at one step earlier
                T prev, next, dump;
                pair_update(om2, om1, o0, o1, c.r, c.g, dump, prev);
                pair_update(oe1, oe, op0, op1, c.r, c.g, next, dump);
                at(s) = prev; at(e) = next;
                T a_old = o1, b_old = oe1;
                int wa = s + 1 + ((s + 1) >> 5), wb = e - 1 + ((e - 1) >> 5);
#pragma unroll 4
                for (int m = 1; m < k; ++m) {
                    const int ra = s + m + 1 + ((s + m + 1) >> 5), rb = e - m - 1 + ((e - m - 1) >> 5);
                    const T a_nxt = sm[ra];
                    const T b_nxt = sm[rb];
                    prev = fma(c.e, (prev - a_old) + (a_nxt - a_old), a_old);
                    sm[wa] = prev;
                    next = fma(c.e, (next - b_old) + (b_nxt - b_old), b_old);
                    sm[wb] = next;
                    a_old = a_nxt; b_old = b_nxt;
                    wa = ra; wb = rb;
                }
            } else if (mine) {
                const int64_t eg = sg + two_k - 1;
                T prev = c.lo, next = c.hi;
                if (sg >= 1) {
                    T lo_, hi_;
                    pair_update_bc(om2, om1, o0, o1, c, sg - 1 == 0, false, lo_, hi_);
                    prev = hi_;
                    if (s >= 0 && s < len) at(s) = prev;
                }
                if (eg >= 1 && eg <= N) {
                    T lo_, hi_;
                    pair_update_bc(oe1, oe, op0, op1, c, false, eg + 1 == N + 1, lo_, hi_);
                    next = lo_;
                    if (e >= 0 && e < len) at(e) = next;
                }
                T a_old = o1, b_old = oe1;
#pragma unroll 1
                for (int m = 1; m < k; ++m) {
                    const int ja = s + m, jb = e - m;
                    const int64_t ia = sg + m, ib = eg - m;
                    const T a_nxt = rd(ja + 1);
                    const T b_nxt = rd(jb - 1);
                    if (ia >= 1 && ia <= N) {
                        prev = fma(c.e, (prev - a_old) + (a_nxt - a_old), a_old);
                        if (ja >= 0 && ja < len) at(ja) = prev;
                    }
                    if (ib >= 1 && ib <= N) {
                        next = fma(c.e, (next - b_old) + (b_nxt - b_old), b_old);
                        if (jb >= 0 && jb < len) at(jb) = next;
                    }
                    a_old = a_nxt; b_old = b_nxt;
                }
            }
            __syncthreads();
        }
        for (int64_t i = v0 + t; i < v1; i += blockDim.x) out[i - 1] = at((int)(i - w0));
        __syncthreads();                                               // the window is reused by the next rod
    }
}

}  // namespace ge
