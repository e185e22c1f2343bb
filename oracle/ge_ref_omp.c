/*
 * ge_ref_omp.c -- ORACLE-SIDE TIMING DRIVER (test infrastructure, NOT the product, NOT the parity oracle).
 *
 * The all-cores leg of the timed CPU baseline ("the oracle timed (a) single thread and
 * (b) an OpenMP parallel-for over the groups within a level -- a separate timed driver; the parity
 * oracle stays scalar").  The paper's own comparison is against an 8-thread C code.
 * The parity oracle is oracle/ge_ref.c and stays scalar and untouched; this file restates the same
 * literal formulas (Eqs (1)-(4) with the prefactor 1/(1+2r), reading R-A1; the 2x2
 * four-point groups of reading R-2D) with the loop over the groups of a level split across threads --
 * the groups of one level are independent of each other for k = 1 (neighbours share
 * nothing but old-level wall nodes).  tests/test_oracle_omp.py pins it to ge_ref.c bit for bit
 * (-ffp-contract=off on both sides, same expressions in the same order).
 *
 * Only bench.py's cpu_baseline leg and tests/ may build, load or call this file.  It shares no code
 * with paper_1310_3422_b200/csrc.  k = 1 only (two-point groups; the BASELINE.json configs).
 */
#include <stdint.h>
#include <stdlib.h>
#include <string.h>
#ifdef _OPENMP
#include <omp.h>
#endif

int ge_omp_threads(void)
{
#ifdef _OPENMP
    return omp_get_max_threads();
#else
    return 1;
#endif
}

/* One level of one rod, k = 1: the pairs (i, i+1), i = 1 + phase (mod 2), in parallel; a pair with a
   boundary member updates its interior member by Eq (1) / Eq (2).
   old_, new_: length N+2, boundary values in [0] and [N+1].  Called from inside a parallel region
   or outside of one (orphaned `omp for`). */
static void level_1d(const double *old_, double *new_, int64_t N, double r, int64_t phase)
{
    const int64_t first = phase ? 0 : 1;            /* left members: first, first+2, ... <= N */
    const int64_t npairs = (N - first) / 2 + 1;
    int64_t m;
#pragma omp for schedule(static)
    for (m = 0; m < npairs; ++m) {
        const int64_t i = first + 2 * m;
        if (i >= 1 && i + 1 <= N) {
            new_[i] = ((r + r * r) * old_[i - 1] + (1.0 - r * r) * old_[i]
                       + (r - r * r) * old_[i + 1] + r * r * old_[i + 2])
                      / (1.0 + 2.0 * r);                                   /* Eq (3) */
            new_[i + 1] = (r * r * old_[i - 1] + (r - r * r) * old_[i]
                           + (1.0 - r * r) * old_[i + 1] + (r + r * r) * old_[i + 2])
                          / (1.0 + 2.0 * r);                               /* Eq (4) */
        } else if (i == 0 && N >= 1) {
            new_[1] = (r * old_[0] + (1.0 - r) * old_[1] + r * old_[2]) / (1.0 + r);        /* Eq (1) */
        } else if (i == N && N >= 1) {
            new_[N] = (r * old_[N + 1] + (1.0 - r) * old_[N] + r * old_[N - 1]) / (1.0 + r); /* Eq (2) */
        }
    }
}

/* `steps` levels of one rod; u: N interior values, overwritten.  Returns 0, or -1 if out of memory. */
int ge_omp_run_1d(double *u, int64_t N, double r, double bc_lo, double bc_hi, int64_t level0, int64_t steps)
{
    double *a = (double *)malloc((size_t)(N + 2) * sizeof(double));
    double *b = (double *)malloc((size_t)(N + 2) * sizeof(double));
    if (!a || !b) { free(a); free(b); return -1; }
    a[0] = bc_lo; a[N + 1] = bc_hi;
    b[0] = bc_lo; b[N + 1] = bc_hi;
    memcpy(a + 1, u, (size_t)N * sizeof(double));
#pragma omp parallel
    {
        double *x = a, *y = b;
        int64_t s;
        for (s = 0; s < steps; ++s) {
            double *t;
            level_1d(x, y, N, r, (level0 + s) & 1);     /* implicit barrier at the end of the omp for */
            t = x; x = y; y = t;
        }
    }
    memcpy(u, (steps & 1) ? b + 1 : a + 1, (size_t)N * sizeof(double));
    free(a); free(b);
    return 0;
}

/* Batched rods (BASELINE.json configs[2]): the rods are independent, one rod per thread at a time. */
int ge_omp_run_batched_1d(double *u, int64_t batch, int64_t N, const double *r, const double *bc_lo,
                          const double *bc_hi, int64_t level0, int64_t steps)
{
    int fail = 0;
    int64_t bb;
#pragma omp parallel for schedule(dynamic, 1)
    for (bb = 0; bb < batch; ++bb) {
        double *a = (double *)malloc((size_t)(N + 2) * sizeof(double));
        double *b = (double *)malloc((size_t)(N + 2) * sizeof(double));
        if (!a || !b) { free(a); free(b); fail = 1; continue; }
        a[0] = bc_lo[bb]; a[N + 1] = bc_hi[bb];
        b[0] = bc_lo[bb]; b[N + 1] = bc_hi[bb];
        memcpy(a + 1, u + bb * N, (size_t)N * sizeof(double));
        {
            double *x = a, *y = b;
            int64_t s, m;
            for (s = 0; s < steps; ++s) {
                const int64_t phase = (level0 + s) & 1;
                const int64_t first = phase ? 0 : 1;
                const double rr = r[bb];
                double *t;
                for (m = first; m <= N; m += 2) {
                    const int64_t i = m;
                    if (i >= 1 && i + 1 <= N) {
                        y[i] = ((rr + rr * rr) * x[i - 1] + (1.0 - rr * rr) * x[i]
                                + (rr - rr * rr) * x[i + 1] + rr * rr * x[i + 2]) / (1.0 + 2.0 * rr);
                        y[i + 1] = (rr * rr * x[i - 1] + (rr - rr * rr) * x[i]
                                    + (1.0 - rr * rr) * x[i + 1] + (rr + rr * rr) * x[i + 2]) / (1.0 + 2.0 * rr);
                    } else if (i == 0 && N >= 1) {
                        y[1] = (rr * x[0] + (1.0 - rr) * x[1] + rr * x[2]) / (1.0 + rr);
                    } else if (i == N && N >= 1) {
                        y[N] = (rr * x[N + 1] + (1.0 - rr) * x[N] + rr * x[N - 1]) / (1.0 + rr);
                    }
                }
                t = x; x = y; y = t;
            }
            memcpy(u + bb * N, x + 1, (size_t)N * sizeof(double));
        }
        free(a); free(b);
    }
    return fail ? -1 : 0;
}

#define AT(a, i, j) ((a)[(size_t)(j) * (size_t)sx + (size_t)(i)])

/* One 2-D level (reading R-2D): the group rows in parallel.  Arrays (Ny+2) x (Nx+2), edges hold the
   boundary values (constant in time; both arrays are initialised with them by the caller). */
static void level_2d(const double *old_, double *new_, int64_t Nx, int64_t Ny, double r, int64_t phase)
{
    const int64_t sx = Nx + 2;
    const double al = 1.0 + 4.0 * r + 2.0 * r * r;
    const double be = r * (1.0 + 2.0 * r);
    const double ga = 2.0 * r * r;
    const double det4 = (1.0 + 2.0 * r) * (1.0 + 4.0 * r);
    const double det2 = (1.0 + r) * (1.0 + 3.0 * r);
    const int64_t g0 = 1 - phase;
    const int64_t nrows = (Ny - g0) / 2 + 1;
    int64_t m;
#pragma omp for schedule(static)
    for (m = 0; m < nrows; ++m) {
        const int64_t gj = g0 + 2 * m;
        int64_t gi;
        for (gi = g0; gi <= Nx; gi += 2) {
            const int x0 = (gi >= 1), x1 = (gi + 1 <= Nx);
            const int y0 = (gj >= 1), y1 = (gj + 1 <= Ny);
            double R[2][2];
            int dx, dy;
            for (dy = 0; dy < 2; ++dy)
                for (dx = 0; dx < 2; ++dx) {
                    const int64_t pi = gi + dx, pj = gj + dy;
                    const int inside = (dx ? x1 : x0) && (dy ? y1 : y0);
                    if (!inside) { R[dy][dx] = 0.0; continue; }
                    R[dy][dx] = (1.0 - 2.0 * r) * AT(old_, pi, pj)
                              + r * AT(old_, pi + (dx ? 1 : -1), pj)
                              + r * AT(old_, pi, pj + (dy ? 1 : -1));
                    if (!(dx ? x0 : x1)) R[dy][dx] += r * AT(old_, pi + (dx ? -1 : 1), pj);
                    if (!(dy ? y0 : y1)) R[dy][dx] += r * AT(old_, pi, pj + (dy ? -1 : 1));
                }
            if (x0 && x1 && y0 && y1) {
                const double Ra = R[0][0], Rb = R[0][1], Rc = R[1][0], Rd = R[1][1];
                AT(new_, gi,     gj)     = (al * Ra + be * Rb + be * Rc + ga * Rd) / det4;
                AT(new_, gi + 1, gj)     = (be * Ra + al * Rb + ga * Rc + be * Rd) / det4;
                AT(new_, gi,     gj + 1) = (be * Ra + ga * Rb + al * Rc + be * Rd) / det4;
                AT(new_, gi + 1, gj + 1) = (ga * Ra + be * Rb + be * Rc + al * Rd) / det4;
            } else if (x0 && x1) {
                const int64_t pj = y0 ? gj : gj + 1;
                const double R1 = R[y0 ? 0 : 1][0], R2 = R[y0 ? 0 : 1][1];
                if (!(y0 || y1)) continue;
                AT(new_, gi,     pj) = ((1.0 + 2.0 * r) * R1 + r * R2) / det2;
                AT(new_, gi + 1, pj) = (r * R1 + (1.0 + 2.0 * r) * R2) / det2;
            } else if (y0 && y1) {
                const int64_t pi = x0 ? gi : gi + 1;
                const double R1 = R[0][x0 ? 0 : 1], R2 = R[1][x0 ? 0 : 1];
                if (!(x0 || x1)) continue;
                AT(new_, pi, gj)     = ((1.0 + 2.0 * r) * R1 + r * R2) / det2;
                AT(new_, pi, gj + 1) = (r * R1 + (1.0 + 2.0 * r) * R2) / det2;
            } else if ((x0 || x1) && (y0 || y1)) {
                const int64_t pi = x0 ? gi : gi + 1, pj = y0 ? gj : gj + 1;
                AT(new_, pi, pj) = R[y0 ? 0 : 1][x0 ? 0 : 1] / (1.0 + 2.0 * r);
            }
        }
    }
}

/* `steps` 2-D levels; u: Ny x Nx interior values, row-major, overwritten; bc = {x_lo, x_hi, y_lo, y_hi}. */
int ge_omp_run_2d(double *u, int64_t Nx, int64_t Ny, double r, const double *bc, int64_t level0, int64_t steps)
{
    const int64_t sx = Nx + 2;
    const size_t tot = (size_t)(Nx + 2) * (size_t)(Ny + 2);
    double *a = (double *)calloc(tot, sizeof(double));
    double *b = (double *)calloc(tot, sizeof(double));
    int64_t i, j;
    if (!a || !b) { free(a); free(b); return -1; }
    for (j = 0; j <= Ny + 1; ++j) { AT(a, 0, j) = bc[0]; AT(a, Nx + 1, j) = bc[1]; }
    for (i = 1; i <= Nx; ++i) { AT(a, i, 0) = bc[2]; AT(a, i, Ny + 1) = bc[3]; }
    for (j = 1; j <= Ny; ++j)
        memcpy(&AT(a, 1, j), u + (size_t)(j - 1) * (size_t)Nx, (size_t)Nx * sizeof(double));
    memcpy(b, a, tot * sizeof(double));                 /* the edges of both levels */
#pragma omp parallel
    {
        double *x = a, *y = b;
        int64_t s;
        for (s = 0; s < steps; ++s) {
            double *t;
            level_2d(x, y, Nx, Ny, r, (level0 + s) & 1);
            t = x; x = y; y = t;
        }
    }
    {
        const double *fin = (steps & 1) ? b : a;
        for (j = 1; j <= Ny; ++j)
            memcpy(u + (size_t)(j - 1) * (size_t)Nx, &AT(fin, 1, j), (size_t)Nx * sizeof(double));
    }
    free(a); free(b);
    return 0;
}
