// ge_window.cuh -- strategy B for NON-CONSTANT problem data: `levels` <= tb levels per HBM
// round trip with a stationary source term and moving boundary values (reading R-N3), or with variable
// diffusivity (reading R-VAR); two-point groups (k = 1), batched rods included.
//
// The register kernels of the constant-coefficient path keep nothing but u; here every node also has a source
// value or every link a coefficient, so a CTA keeps a window of the rod in shared memory -- two copies of u
// (ping-pong: one CTA barrier per level), the window of tau*f or of the link numbers -- and marches it like the
// per-level kernels do (ge_level_src.cuh, ge_level_var.cuh: the same expressions).  A pair reads u_{i-1} .. u_{i+2}
// (PAPER.md:96-101), so what a cut end of the window spoils moves inward by two nodes per level: halo = 2 tb + 2.
// A window end that is the rod's end holds the Dirichlet node; with moving boundary values the new level's value
// is written there before the level is marched (a truncated pair takes the NEW value, an old-level read the OLD one).
#pragma once
#include "ge_common.cuh"

namespace ge {

constexpr int kWinThreads = 256;
constexpr int kWinNodes = 2048;          // nodes of a window (shared memory: 3 arrays of kWinNodes + 2 values)

struct WinGeom {
    int tb, halo, valid;
    int64_t tiles;
};
inline WinGeom win_geom(int tb, int64_t nx) {
    WinGeom g;
    g.tb = tb;
    g.halo = 2 * tb + 2;
    int64_t valid = kWinNodes - 2 * g.halo;
    valid -= valid % 2;
    if (valid > nx) valid = nx + (nx & 1);
    g.valid = valid >= 2 ? (int)valid : 0;
    g.tiles = g.valid > 0 ? (nx + g.valid - 1) / g.valid : 0;
    return g;
}
template <typename T>
inline size_t win_smem() { return (size_t)3 * (kWinNodes + 4) * sizeof(T); }

// SRC: src = tau*f, [batch][nx], stationary; bc = [batch][nlev+1][2] boundary values (lo, hi) at the run's levels,
//      bc_lev = index of the first level of this launch, bc_stride = nlev + 1.
// VAR: rl = link numbers, [batch][nx+1]; boundary values constant (the plan's).
template <typename T, bool SRC, bool VAR>
__global__ void __launch_bounds__(kWinThreads)
ge1d_window_kernel(const T* __restrict__ uin, T* __restrict__ uout, const T* __restrict__ src, const T* __restrict__ rl,
                   const T* __restrict__ bc, int64_t bc_lev, int64_t bc_stride, int64_t nx, int64_t batch,
                   const Coef1<T>* __restrict__ coef, const WinGeom g, int phase0, int levels) {
    extern __shared__ __align__(16) unsigned char win_smem_raw[];
    T* xa = reinterpret_cast<T*>(win_smem_raw);
    T* xb = xa + kWinNodes + 4;
    T* aux = xb + kWinNodes + 4;                   // SRC: tau*f of node w0+j at [j]; VAR: link (w0+j, w0+j+1) at [j]
    const int64_t N = nx;
    const int t = threadIdx.x;
    const int64_t v0 = 1 + (int64_t)blockIdx.x * g.valid;
    const int64_t v1 = v0 + g.valid < N + 1 ? v0 + g.valid : N + 1;
    int64_t w0 = v0 - g.halo > 0 ? v0 - g.halo : 0;
    w0 -= w0 & 1;                                  // even: the pair pattern of the window is the global one
    const int64_t w1 = v1 + g.halo < N + 2 ? v1 + g.halo : N + 2;
    const int len = (int)(w1 - w0);                // nodes w0 .. w1-1
    auto cp = [&](T* dst, const T* gsrc) {
        const uint32_t d32 = (uint32_t)__cvta_generic_to_shared(dst);
        if constexpr (sizeof(T) == 8) asm volatile("cp.async.ca.shared.global [%0], [%1], 8;" ::"r"(d32), "l"(gsrc) : "memory");
        else                          asm volatile("cp.async.ca.shared.global [%0], [%1], 4;" ::"r"(d32), "l"(gsrc) : "memory");
    };
    for (int64_t rod = blockIdx.y; rod < batch; rod += gridDim.y) {
        const Coef1<T> c = coef[rod];
        const T* __restrict__ in = uin + rod * nx;
        T* __restrict__ out = uout + rod * nx;
        const T* __restrict__ bcr = SRC ? bc + (rod * bc_stride + bc_lev) * 2 : nullptr;
        T lo_old = SRC ? bcr[0] : c.lo, hi_old = SRC ? bcr[1] : c.hi;
        for (int j = t; j < len; j += kWinThreads) {
            const int64_t i = w0 + j;
            if (i >= 1 && i <= N) {
                cp(xa + j, in + (i - 1));
                if constexpr (SRC) { if (src) cp(aux + j, src + rod * nx + (i - 1)); else aux[j] = T(0); }
            } else {
                xa[j] = i == 0 ? lo_old : hi_old;
                if constexpr (SRC) aux[j] = T(0);
            }
            if constexpr (VAR) { if (i <= N) cp(aux + j, rl + rod * (nx + 1) + i); else aux[j] = T(1); }
        }
        asm volatile("cp.async.wait_all;" ::: "memory");
        __syncthreads();
        T* x = xa; T* y = xb;
#pragma unroll 1
        for (int lev = 0; lev < levels; ++lev) {
            const int ph = (phase0 + lev) & 1;
            const T lo_new = SRC ? bcr[2 * (lev + 1)] : c.lo, hi_new = SRC ? bcr[2 * (lev + 1) + 1] : c.hi;
            if (t == 0) {                          // Dirichlet nodes of the new level (cut ends are stale halo)
                if (w0 == 0) y[0] = lo_new;
                if (w1 == N + 2) y[len - 1] = hi_new;
            }
            // left members at window positions of parity 1 - ph (w0 is even; phase 0 pairs nodes (1,2),(3,4),...)
            if (w0 > 0 && w1 < N + 2) {
                // a window without a rod end (CTA-uniform): no Dirichlet tests, 32-bit indices; the pairs that would
                // read beyond the window's ends are left alone (stale halo)
                int j = (1 - ph) + 2 * t;
                if (j == 0) j += 2 * kWinThreads;
#pragma unroll 2
                for (; j + 2 < len; j += 2 * kWinThreads) {
                    const T a = x[j - 1], b = x[j], cc = x[j + 1], d = x[j + 2];
                    T p, q, gg;
                    if constexpr (VAR) {
                        const T rm = aux[j];
                        p = fma(aux[j - 1], a - b, b);
                        q = fma(aux[j + 1], d - cc, cc);
                        gg = rm / fma(T(2), rm, T(1));
                    } else {
                        p = fma(c.r, a - b, b) + aux[j];
                        q = fma(c.r, d - cc, cc) + aux[j + 1];
                        gg = c.g;
                    }
                    const T tt = q - p;
                    y[j] = fma(gg, tt, p);
                    y[j + 1] = fma(-gg, tt, q);
                }
            } else
            for (int j = (1 - ph) + 2 * t; j < len; j += 2 * kWinThreads) {
                const int64_t i = w0 + j;          // node of the left member
                if (i > N) break;
                if (j + 1 >= len) { continue; }    // the right member lies beyond a cut end: stale halo
                const bool b_bc = i == 0, c_bc = i + 1 == N + 1;
                const T a = j > 0 ? x[j - 1] : x[j];
                const T b = x[j], cc = x[j + 1];
                const T d = j + 2 < len ? x[j + 2] : cc;
                T p, q, gg;
                if constexpr (VAR) {
                    const T rm = aux[j];
                    p = b_bc ? lo_new : fma(j > 0 ? aux[j - 1] : aux[j], a - b, b);
                    q = c_bc ? hi_new : fma(aux[j + 1], d - cc, cc);
                    gg = rm / ((b_bc || c_bc) ? T(1) + rm : fma(T(2), rm, T(1)));
                } else {
                    p = b_bc ? lo_new : fma(c.r, a - b, b) + aux[j];
                    q = c_bc ? hi_new : fma(c.r, d - cc, cc) + aux[j + 1];
                    gg = (b_bc || c_bc) ? c.e : c.g;
                }
                const T tt = q - p;
                if (!b_bc) y[j] = fma(gg, tt, p);
                if (!c_bc) y[j + 1] = fma(-gg, tt, q);
            }
            __syncthreads();
            T* s = x; x = y; y = s;
        }
        for (int64_t i = v0 + t; i < v1; i += kWinThreads) out[i - 1] = x[(int)(i - w0)];
        __syncthreads();                           // the window is reused by the next rod
    }
}

}  // namespace ge
