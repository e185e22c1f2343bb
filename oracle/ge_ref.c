/*
 * ge_ref.c -- ORACLE (test infrastructure, NOT the product).
 *
 * Plain, slow, scalar fp64 CPU statement of the group-explicit (GE) scheme of
 * arXiv 1310.3422 for u_t = u_xx (and the 2x2-group 2-D reading for
 * u_t = u_xx + u_yy).  Only tests/, __graft_entry__.smoke() and bench.py's
 * cpu_baseline / --impl reference legs may build, load or call this file.
 * It shares no code with paper_1310_3422_b200/csrc: the formulas below are
 * written literally as the paper prints them (with the division), never in
 * the factored form the CUDA kernels use.
 *
 * Notation: N interior nodes 1..N, nodes 0 and N+1 are
 * the Dirichlet boundary (h = 1/(N+1)); r = tau/h^2
 * (PAPER.md:73); k = sub-domain length; level = one advance by
 * tau; phase = level mod 2 (the paper's "first row"/"second row",
 * PAPER.md:140-148).  Arrays passed to the *_level_* functions carry the
 * boundary nodes: 1-D length N+2, 2-D (N_y+2) x (N_x+2) row-major.
 *
 * Parity pins (tests/test_oracle_*.py): P1 2x2 solve identity, P2 invariants,
 * P3/P9 exact-rational worked examples (tests/golden), P4 dense A^-1 B brute
 * force from the implicit statement, P5 spectral radius of the two-level
 * cycle, P6/P7 convergence to e^{-pi^2 t} sin(pi x), P8 Saul'yev special case.
 * The 2-D functions follow DESIGN.md reading R-2D (PAPER.md defines no 2-D
 * scheme; PAPER.md:134, :228 only claim the extension) and are pinned by
 * P2, P4, P5, P6, P8, P9 only: "parity unpinned by the paper" for 2-D.
 */
#include <stdint.h>
#include <stdlib.h>
#include <string.h>

/* non-negative remainder */
static int64_t pmod(int64_t a, int64_t m) {
    int64_t x = a % m;
    return x < 0 ? x + m : x;
}

/*
 * One level in 1-D for any k >= 1.
 *
 * Class of node i: c(i) = (i - phase*k) mod 2k
 *   c == 2k-1 : left member of the confluence pair (i, i+1)   -> Eq (3)
 *   c == 0    : right member of the pair (i-1, i)             -> Eq (4)
 *   1..k-1    : Saul'yev A, Eq (1), ascending i (uses new[i-1])
 *   k..2k-2   : Saul'yev B, Eq (2), descending i (uses new[i+1])
 * Prefactor of Eqs (3),(4): 1/(1+2r) (the printed "3" is an extraction
 * artefact: the four weights sum to 1+2r; reading R-A1).
 * A pair with a boundary member is not solved as a pair: its interior member
 * takes Eq (1) (partner node 0) or Eq (2) (partner node N+1) with the boundary
 * value as the new-level neighbour ("preinitialized").
 *
 * old_, new_: length N+2; old_[0], old_[N+1] hold the boundary values, which
 * are copied to new_ (constant in time).
 */
void ge_ref_level_1d(const double *old_, double *new_, int64_t N, double r,
                     int64_t k, int64_t phase)
{
    const int64_t two_k = 2 * k;
    int64_t i;
    new_[0] = old_[0];
    new_[N + 1] = old_[N + 1];

    /* first: confluence pairs, any order */
    for (i = 0; i <= N; ++i) {
        if (pmod(i - phase * k, two_k) != two_k - 1) continue;
        /* i is a left member, i+1 the right member */
        if (i >= 1 && i + 1 <= N) {
            new_[i] = ((r + r * r) * old_[i - 1] + (1.0 - r * r) * old_[i]
                       + (r - r * r) * old_[i + 1] + r * r * old_[i + 2])
                      / (1.0 + 2.0 * r);                                   /* Eq (3) */
            new_[i + 1] = (r * r * old_[i - 1] + (r - r * r) * old_[i]
                           + (1.0 - r * r) * old_[i + 1] + (r + r * r) * old_[i + 2])
                          / (1.0 + 2.0 * r);                               /* Eq (4) */
        } else if (i == 0 && N >= 1) {
            /* pair (0,1): node 0 is boundary -> node 1 by Eq (1) */
            new_[1] = (r * new_[0] + (1.0 - r) * old_[1] + r * old_[2]) / (1.0 + r);
        } else if (i == N && N >= 1) {
            /* pair (N,N+1): node N+1 is boundary -> node N by Eq (2) */
            new_[N] = (r * new_[N + 1] + (1.0 - r) * old_[N] + r * old_[N - 1]) / (1.0 + r);
        }
    }
    /* second: Eq (1) nodes, ascending */
    for (i = 1; i <= N; ++i) {
        int64_t c = pmod(i - phase * k, two_k);
        if (c >= 1 && c <= k - 1)
            new_[i] = (r * new_[i - 1] + (1.0 - r) * old_[i] + r * old_[i + 1]) / (1.0 + r);
    }
    /* third: Eq (2) nodes, descending */
    for (i = N; i >= 1; --i) {
        int64_t c = pmod(i - phase * k, two_k);
        if (c >= k && c <= two_k - 2)
            new_[i] = (r * new_[i + 1] + (1.0 - r) * old_[i] + r * old_[i - 1]) / (1.0 + r);
    }
}

/*
 * One level in 1-D with a source term and time-dependent boundary values
 * (reading R-N3; SURVEY.md 8(f) NEXT-3 -- the paper's model problem has
 * neither; PAPER.md:37 only mentions the diffusion step inside
 * an operator splitting):   u_t = u_xx + f(x,t),  u(0,t) = lo(t),  u(1,t) = hi(t).
 * Saul'yev's asymmetric equations gain tau*f at their node,
 *   Eq (1): (1+r) new_i = r new_{i-1} + (1-r) old_i + r old_{i+1} + s_i
 *   Eq (2): (1+r) new_i = r new_{i+1} + (1-r) old_i + r old_{i-1} + s_i
 * and a confluence pair is the 2x2 system of Eq (2) at i with Eq (1) at i+1,
 * whose solution is the bracket of Eq (3)/(4) plus (1+r) s_i + r s_{i+1}
 * (resp. r s_i + (1+r) s_{i+1}), all over 1+2r.  Old-level reads of a boundary
 * node take its OLD value (old_[0], old_[N+1]); the new-level neighbour of a
 * truncated pair or of a sweep is the NEW value (lo_new, hi_new).
 * s: length N+2, s[i] = tau * f(x_i, t*) for i = 1..N (t* is the caller's
 * choice), or NULL for no source.
 */
void ge_ref_level_1d_src(const double *old_, double *new_, int64_t N, double r,
                         int64_t k, int64_t phase, const double *s,
                         double lo_new, double hi_new)
{
    const int64_t two_k = 2 * k;
    int64_t i;
    new_[0] = lo_new;
    new_[N + 1] = hi_new;
    for (i = 0; i <= N; ++i) {
        if (pmod(i - phase * k, two_k) != two_k - 1) continue;
        if (i >= 1 && i + 1 <= N) {
            const double si = s ? s[i] : 0.0, sj = s ? s[i + 1] : 0.0;
            new_[i] = ((r + r * r) * old_[i - 1] + (1.0 - r * r) * old_[i]
                       + (r - r * r) * old_[i + 1] + r * r * old_[i + 2]
                       + (1.0 + r) * si + r * sj) / (1.0 + 2.0 * r);
            new_[i + 1] = (r * r * old_[i - 1] + (r - r * r) * old_[i]
                           + (1.0 - r * r) * old_[i + 1] + (r + r * r) * old_[i + 2]
                           + r * si + (1.0 + r) * sj) / (1.0 + 2.0 * r);
        } else if (i == 0 && N >= 1) {
            new_[1] = (r * new_[0] + (1.0 - r) * old_[1] + r * old_[2] + (s ? s[1] : 0.0)) / (1.0 + r);
        } else if (i == N && N >= 1) {
            new_[N] = (r * new_[N + 1] + (1.0 - r) * old_[N] + r * old_[N - 1] + (s ? s[N] : 0.0)) / (1.0 + r);
        }
    }
    for (i = 1; i <= N; ++i) {
        int64_t c = pmod(i - phase * k, two_k);
        if (c >= 1 && c <= k - 1)
            new_[i] = (r * new_[i - 1] + (1.0 - r) * old_[i] + r * old_[i + 1] + (s ? s[i] : 0.0)) / (1.0 + r);
    }
    for (i = N; i >= 1; --i) {
        int64_t c = pmod(i - phase * k, two_k);
        if (c >= k && c <= two_k - 2)
            new_[i] = (r * new_[i + 1] + (1.0 - r) * old_[i] + r * old_[i - 1] + (s ? s[i] : 0.0)) / (1.0 + r);
    }
}

/*
 * `steps` levels of one rod starting at level counter `level0` (phase =
 * level mod 2, phase 0 first: DESIGN.md reading R-A3).  u holds the N
 * interior values and is overwritten by the final level.  Returns 0, or -1 if
 * out of memory.
 */
int ge_ref_run_1d(double *u, int64_t N, double r, int64_t k, double bc_lo,
                  double bc_hi, int64_t level0, int64_t steps)
{
    double *a = (double *)malloc((size_t)(N + 2) * sizeof(double));
    double *b = (double *)malloc((size_t)(N + 2) * sizeof(double));
    int64_t s;
    if (!a || !b) { free(a); free(b); return -1; }
    a[0] = bc_lo; a[N + 1] = bc_hi;
    memcpy(a + 1, u, (size_t)N * sizeof(double));
    for (s = 0; s < steps; ++s) {
        double *t;
        ge_ref_level_1d(a, b, N, r, k, pmod(level0 + s, 2));
        t = a; a = b; b = t;
    }
    memcpy(u, a + 1, (size_t)N * sizeof(double));
    free(a); free(b);
    return 0;
}

/*
 * Batched rods (BASELINE.json configs[2]): rod b has its own r[b], bc_lo[b],
 * bc_hi[b]; u is [batch][N] row-major, interior values only.
 */
int ge_ref_run_batched_1d(double *u, int64_t batch, int64_t N, const double *r,
                          int64_t k, const double *bc_lo, const double *bc_hi,
                          int64_t level0, int64_t steps)
{
    int64_t b;
    for (b = 0; b < batch; ++b) {
        int rc = ge_ref_run_1d(u + b * N, N, r[b], k, bc_lo[b], bc_hi[b], level0, steps);
        if (rc) return rc;
    }
    return 0;
}

/*
 * One level in 2-D, 2x2 four-point groups (reading R-2D).
 *
 * Nodes (i,j), i = 0..Nx+1 along x (fastest), j = 0..Ny+1 along y; interior
 * 1..N; edges Dirichlet; corner nodes are never read.  Group anchors
 * (lower-left member) at i == 1+phase, j == 1+phase (mod 2): phase 0 anchors
 * 1,3,5,...; phase 1 anchors 0,2,4,... (diagonal shift), groups sticking out
 * over an edge keep only their interior members.
 *
 * For an interior member P with in-group neighbours G (new level) and
 * out-of-group neighbours O (old level):
 *     (1+2r) new_P - r sum_G new_G = R_P := (1-2r) old_P + r sum_O old_O
 * where a boundary in-group neighbour contributes r*beta to the right side.
 *
 * Full group a=(i,j) b=(i+1,j) c=(i,j+1) d=(i+1,j+1):
 *   new = M (R_a,R_b,R_c,R_d)^T / ((1+2r)(1+4r)),
 *   M = [[al,be,be,ga],[be,al,ga,be],[be,ga,al,be],[ga,be,be,al]],
 *   al = 1+4r+2r^2, be = r(1+2r), ga = 2r^2.
 * Edge group (two interior members adjacent along the edge):
 *   new_1 = ((1+2r) R_1 + r R_2) / ((1+r)(1+3r)), symmetric for new_2.
 * Corner group (one interior member): new = R / (1+2r).
 */
#define AT(a, i, j) ((a)[(size_t)(j) * (size_t)sx + (size_t)(i)])

void ge_ref_level_2d(const double *old_, double *new_, int64_t Nx, int64_t Ny,
                     double r, int64_t phase)
{
    const int64_t sx = Nx + 2;
    const double al = 1.0 + 4.0 * r + 2.0 * r * r;
    const double be = r * (1.0 + 2.0 * r);
    const double ga = 2.0 * r * r;
    const double det4 = (1.0 + 2.0 * r) * (1.0 + 4.0 * r);
    const double det2 = (1.0 + r) * (1.0 + 3.0 * r);
    int64_t i, j, gi, gj;

    /* boundary nodes are constant in time */
    for (i = 0; i <= Nx + 1; ++i) { AT(new_, i, 0) = AT(old_, i, 0); AT(new_, i, Ny + 1) = AT(old_, i, Ny + 1); }
    for (j = 0; j <= Ny + 1; ++j) { AT(new_, 0, j) = AT(old_, 0, j); AT(new_, Nx + 1, j) = AT(old_, Nx + 1, j); }

    for (gj = 1 - phase; gj <= Ny; gj += 2) {
        for (gi = 1 - phase; gi <= Nx; gi += 2) {
            /* members: (gi,gj) (gi+1,gj) (gi,gj+1) (gi+1,gj+1); which are interior? */
            const int x0 = (gi >= 1), x1 = (gi + 1 <= Nx);
            const int y0 = (gj >= 1), y1 = (gj + 1 <= Ny);
            /* right-hand sides: out-of-group neighbours at the old level.  For
               member (gi+dx, gj+dy) the out-of-group x-neighbour is at
               gi+dx + (dx ? +1 : -1), likewise in y. */
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
                    /* in-group neighbour that is a boundary node: known value */
                    if (!(dx ? x0 : x1)) R[dy][dx] += r * AT(old_, pi + (dx ? -1 : 1), pj);
                    if (!(dy ? y0 : y1)) R[dy][dx] += r * AT(old_, pi, pj + (dy ? -1 : 1));
                }
            if (x0 && x1 && y0 && y1) {
                const double Ra = R[0][0], Rb = R[0][1], Rc = R[1][0], Rd = R[1][1];
                AT(new_, gi,     gj)     = (al * Ra + be * Rb + be * Rc + ga * Rd) / det4;
                AT(new_, gi + 1, gj)     = (be * Ra + al * Rb + ga * Rc + be * Rd) / det4;
                AT(new_, gi,     gj + 1) = (be * Ra + ga * Rb + al * Rc + be * Rd) / det4;
                AT(new_, gi + 1, gj + 1) = (ga * Ra + be * Rb + be * Rc + al * Rd) / det4;
            } else if (x0 && x1) {            /* one interior row: members along x */
                const int64_t pj = y0 ? gj : gj + 1;
                const double R1 = R[y0 ? 0 : 1][0], R2 = R[y0 ? 0 : 1][1];
                if (!(y0 || y1)) continue;
                AT(new_, gi,     pj) = ((1.0 + 2.0 * r) * R1 + r * R2) / det2;
                AT(new_, gi + 1, pj) = (r * R1 + (1.0 + 2.0 * r) * R2) / det2;
            } else if (y0 && y1) {            /* one interior column: members along y */
                const int64_t pi = x0 ? gi : gi + 1;
                const double R1 = R[0][x0 ? 0 : 1], R2 = R[1][x0 ? 0 : 1];
                if (!(x0 || x1)) continue;
                AT(new_, pi, gj)     = ((1.0 + 2.0 * r) * R1 + r * R2) / det2;
                AT(new_, pi, gj + 1) = (r * R1 + (1.0 + 2.0 * r) * R2) / det2;
            } else if ((x0 || x1) && (y0 || y1)) {   /* single interior member */
                const int64_t pi = x0 ? gi : gi + 1, pj = y0 ? gj : gj + 1;
                AT(new_, pi, pj) = R[y0 ? 0 : 1][x0 ? 0 : 1] / (1.0 + 2.0 * r);
            }
        }
    }
}

/*
 * `steps` levels in 2-D.  u: Ny x Nx interior values, row-major [j][i],
 * overwritten by the final level.  bc = {x_lo, x_hi, y_lo, y_hi}: the constant
 * value on the edges i=0, i=Nx+1, j=0, j=Ny+1.
 */
int ge_ref_run_2d(double *u, int64_t Nx, int64_t Ny, double r, const double *bc,
                  int64_t level0, int64_t steps)
{
    const int64_t sx = Nx + 2;
    const size_t tot = (size_t)(Nx + 2) * (size_t)(Ny + 2);
    double *a = (double *)calloc(tot, sizeof(double));
    double *b = (double *)calloc(tot, sizeof(double));
    int64_t i, j, s;
    if (!a || !b) { free(a); free(b); return -1; }
    for (j = 0; j <= Ny + 1; ++j) { AT(a, 0, j) = bc[0]; AT(a, Nx + 1, j) = bc[1]; }
    for (i = 1; i <= Nx; ++i) { AT(a, i, 0) = bc[2]; AT(a, i, Ny + 1) = bc[3]; }
    for (j = 1; j <= Ny; ++j)
        memcpy(&AT(a, 1, j), u + (size_t)(j - 1) * (size_t)Nx, (size_t)Nx * sizeof(double));
    for (s = 0; s < steps; ++s) {
        double *t;
        ge_ref_level_2d(a, b, Nx, Ny, r, pmod(level0 + s, 2));
        t = a; a = b; b = t;
    }
    for (j = 1; j <= Ny; ++j)
        memcpy(u + (size_t)(j - 1) * (size_t)Nx, &AT(a, 1, j), (size_t)Nx * sizeof(double));
    free(a); free(b);
    return 0;
}

/*
 * One level in 3-D, 2x2x2 eight-point groups (reading R-3D; SURVEY.md
 * 8(f) NEXT-4 -- the paper only claims "capacity of extension to higher order
 * dimensions").  The construction is that of the 2-D
 * reading: group anchors at (1+phase) mod 2 in every axis (shift (1,1,1)
 * between levels), in-group links at the new level, out-of-group links at the
 * old level; for an interior member P with its three in-group neighbours G and
 * its three out-of-group neighbours O
 *     (1+3r) new_P - r sum_G new_G = (1-3r) old_P + r sum_O old_O ,
 * a boundary in-group neighbour contributing r*beta to the right side.  Groups
 * cut by a face, an edge or a corner keep their interior members (4, 2, 1).
 * The m x m system of a group (m <= 8) is solved by plain Gaussian elimination
 * with partial pivoting -- no closed form is used here.
 *
 * Arrays: (Nz+2) x (Ny+2) x (Nx+2), x fastest; the six faces hold the boundary
 * values (constant in time), edge and corner nodes of the box are never read.
 */
#define AT3(a, i, j, k) ((a)[((size_t)(k) * (size_t)sy + (size_t)(j)) * (size_t)sx + (size_t)(i)])

static void solve_small(int m, double A[8][8], double *b)
{
    int c, rr, cc;
    for (c = 0; c < m; ++c) {
        int piv = c;
        double best = A[c][c] < 0 ? -A[c][c] : A[c][c];
        for (rr = c + 1; rr < m; ++rr) {
            double v = A[rr][c] < 0 ? -A[rr][c] : A[rr][c];
            if (v > best) { best = v; piv = rr; }
        }
        if (piv != c) {
            double t;
            for (cc = 0; cc < m; ++cc) { t = A[c][cc]; A[c][cc] = A[piv][cc]; A[piv][cc] = t; }
            t = b[c]; b[c] = b[piv]; b[piv] = t;
        }
        for (rr = c + 1; rr < m; ++rr) {
            const double f = A[rr][c] / A[c][c];
            for (cc = c; cc < m; ++cc) A[rr][cc] -= f * A[c][cc];
            b[rr] -= f * b[c];
        }
    }
    for (c = m - 1; c >= 0; --c) {
        double s = b[c];
        for (cc = c + 1; cc < m; ++cc) s -= A[c][cc] * b[cc];
        b[c] = s / A[c][c];
    }
}

void ge_ref_level_3d(const double *old_, double *new_, int64_t Nx, int64_t Ny, int64_t Nz,
                     double r, int64_t phase)
{
    const int64_t sx = Nx + 2, sy = Ny + 2;
    const int64_t N[3] = {Nx, Ny, Nz};
    int64_t g[3];
    memcpy(new_, old_, (size_t)(Nx + 2) * (size_t)(Ny + 2) * (size_t)(Nz + 2) * sizeof(double));
    for (g[2] = 1 - phase; g[2] <= Nz; g[2] += 2)
        for (g[1] = 1 - phase; g[1] <= Ny; g[1] += 2)
            for (g[0] = 1 - phase; g[0] <= Nx; g[0] += 2) {
                int idx[8], m = 0, d, q, ax;
                double A[8][8], b[8];
                int64_t pos[8][3];
                for (d = 0; d < 8; ++d) {                 /* member d: offsets (d&1, d>>1&1, d>>2&1) */
                    int inside = 1;
                    for (ax = 0; ax < 3; ++ax) {
                        const int64_t p = g[ax] + ((d >> ax) & 1);
                        if (p < 1 || p > N[ax]) inside = 0;
                    }
                    idx[d] = inside ? m : -1;
                    if (inside) {
                        for (ax = 0; ax < 3; ++ax) pos[m][ax] = g[ax] + ((d >> ax) & 1);
                        ++m;
                    }
                }
                if (m == 0) continue;
                for (d = 0; d < 8; ++d) {
                    int row;
                    int64_t p[3];
                    if (idx[d] < 0) continue;
                    row = idx[d];
                    for (ax = 0; ax < 3; ++ax) p[ax] = g[ax] + ((d >> ax) & 1);
                    for (q = 0; q < m; ++q) A[row][q] = 0.0;
                    A[row][row] = 1.0 + 3.0 * r;
                    b[row] = (1.0 - 3.0 * r) * AT3(old_, p[0], p[1], p[2]);
                    for (ax = 0; ax < 3; ++ax) {
                        const int bit = (d >> ax) & 1;
                        int64_t in[3] = {p[0], p[1], p[2]}, out[3] = {p[0], p[1], p[2]};
                        const int partner = d ^ (1 << ax);
                        in[ax] += bit ? -1 : 1;           /* in-group neighbour along this axis  */
                        out[ax] += bit ? 1 : -1;          /* out-of-group neighbour              */
                        b[row] += r * AT3(old_, out[0], out[1], out[2]);
                        if (idx[partner] >= 0) A[row][idx[partner]] -= r;
                        else b[row] += r * AT3(old_, in[0], in[1], in[2]);   /* boundary node: known */
                    }
                }
                solve_small(m, A, b);
                for (q = 0; q < m; ++q) AT3(new_, pos[q][0], pos[q][1], pos[q][2]) = b[q];
            }
}

/*
 * `steps` levels in 3-D.  u: Nz x Ny x Nx interior values, [k][j][i], overwritten
 * by the final level.  bc = {x_lo, x_hi, y_lo, y_hi, z_lo, z_hi}.
 */
int ge_ref_run_3d(double *u, int64_t Nx, int64_t Ny, int64_t Nz, double r, const double *bc,
                  int64_t level0, int64_t steps)
{
    const int64_t sx = Nx + 2, sy = Ny + 2;
    const size_t tot = (size_t)(Nx + 2) * (size_t)(Ny + 2) * (size_t)(Nz + 2);
    double *a = (double *)calloc(tot, sizeof(double));
    double *b = (double *)calloc(tot, sizeof(double));
    int64_t i, j, k, s;
    if (!a || !b) { free(a); free(b); return -1; }
    for (k = 0; k <= Nz + 1; ++k)
        for (j = 0; j <= Ny + 1; ++j)
            for (i = 0; i <= Nx + 1; ++i) {
                double v = 0.0;
                const int onx = (i == 0 || i == Nx + 1), ony = (j == 0 || j == Ny + 1), onz = (k == 0 || k == Nz + 1);
                if (onx + ony + onz == 0) v = u[((size_t)(k - 1) * (size_t)Ny + (size_t)(j - 1)) * (size_t)Nx + (size_t)(i - 1)];
                else if (onx + ony + onz == 1)
                    v = onx ? bc[i == 0 ? 0 : 1] : (ony ? bc[j == 0 ? 2 : 3] : bc[k == 0 ? 4 : 5]);
                AT3(a, i, j, k) = v;
            }
    for (s = 0; s < steps; ++s) {
        double *t;
        ge_ref_level_3d(a, b, Nx, Ny, Nz, r, pmod(level0 + s, 2));
        t = a; a = b; b = t;
    }
    for (k = 1; k <= Nz; ++k)
        for (j = 1; j <= Ny; ++j)
            memcpy(u + ((size_t)(k - 1) * (size_t)Ny + (size_t)(j - 1)) * (size_t)Nx, &AT3(a, 1, j, k),
                   (size_t)Nx * sizeof(double));
    free(a); free(b);
    return 0;
}

/*
 * One level in 1-D with VARIABLE DIFFUSIVITY (reading R-VAR; SURVEY.md 8(f) NEXT-3 -- the paper's
 * model problem has a constant coefficient; PAPER.md:37 names diffusion steps inside an
 * operator splitting of full transport equations as the use):   u_t = (a(x) u_x)_x  in flux form,
 *     (u_i^{n+1} - u_i^n)/tau = [ a_{i+1/2} (u_{i+1} - u_i) - a_{i-1/2} (u_i - u_{i-1}) ] / h^2 ,
 * with one number per LINK:  rl[j] = tau a_{j+1/2} / h^2 > 0 for the link between nodes j and j+1, j = 0..N.
 * Saul'yev's asymmetric equations take the flux through one link at the new level and through the other at
 * the old level:
 *   Eq (1) (ascending):  (1 + rl[i-1]) new_i = rl[i-1] new_{i-1} + (1 - rl[i]) old_i + rl[i] old_{i+1}
 *   Eq (2) (descending): (1 + rl[i])   new_i = rl[i] new_{i+1} + (1 - rl[i-1]) old_i + rl[i-1] old_{i-1}
 * and a confluence pair (i, i+1) is Eq (2) at i coupled with Eq (1) at i+1 -- its inner link rm = rl[i] at
 * the new level, its outer links rl[i-1], rl[i+1] at the old level:
 *   (1 + rm) new_i - rm new_{i+1} = p := (1 - rl[i-1]) old_i + rl[i-1] old_{i-1}
 *   -rm new_i + (1 + rm) new_{i+1} = q := (1 - rl[i+1]) old_{i+1} + rl[i+1] old_{i+2}
 * whose solution is written out below (determinant 1 + 2 rm).  With every rl[j] = r these are Eqs (1)-(4)
 * of the paper.  Node classes, sweep order and boundary truncation are those of ge_ref_level_1d.
 * old_, new_: length N+2 with the boundary values in [0] and [N+1]; rl: length N+1.
 */
void ge_ref_level_1d_var(const double *old_, double *new_, int64_t N, const double *rl,
                         int64_t k, int64_t phase)
{
    const int64_t two_k = 2 * k;
    int64_t i;
    new_[0] = old_[0];
    new_[N + 1] = old_[N + 1];
    for (i = 0; i <= N; ++i) {
        if (pmod(i - phase * k, two_k) != two_k - 1) continue;
        if (i >= 1 && i + 1 <= N) {
            const double rm = rl[i];
            const double p = (1.0 - rl[i - 1]) * old_[i] + rl[i - 1] * old_[i - 1];
            const double q = (1.0 - rl[i + 1]) * old_[i + 1] + rl[i + 1] * old_[i + 2];
            new_[i] = ((1.0 + rm) * p + rm * q) / (1.0 + 2.0 * rm);
            new_[i + 1] = (rm * p + (1.0 + rm) * q) / (1.0 + 2.0 * rm);
        } else if (i == 0 && N >= 1) {
            new_[1] = (rl[0] * new_[0] + (1.0 - rl[1]) * old_[1] + rl[1] * old_[2]) / (1.0 + rl[0]);
        } else if (i == N && N >= 1) {
            new_[N] = (rl[N] * new_[N + 1] + (1.0 - rl[N - 1]) * old_[N] + rl[N - 1] * old_[N - 1]) / (1.0 + rl[N]);
        }
    }
    for (i = 1; i <= N; ++i) {
        int64_t c = pmod(i - phase * k, two_k);
        if (c >= 1 && c <= k - 1)
            new_[i] = (rl[i - 1] * new_[i - 1] + (1.0 - rl[i]) * old_[i] + rl[i] * old_[i + 1]) / (1.0 + rl[i - 1]);
    }
    for (i = N; i >= 1; --i) {
        int64_t c = pmod(i - phase * k, two_k);
        if (c >= k && c <= two_k - 2)
            new_[i] = (rl[i] * new_[i + 1] + (1.0 - rl[i - 1]) * old_[i] + rl[i - 1] * old_[i - 1]) / (1.0 + rl[i]);
    }
}

/* `steps` levels with variable diffusivity; u: N interior values, overwritten; rl: N+1 link numbers. */
int ge_ref_run_1d_var(double *u, int64_t N, const double *rl, int64_t k, double bc_lo, double bc_hi,
                      int64_t level0, int64_t steps)
{
    double *a = (double *)malloc((size_t)(N + 2) * sizeof(double));
    double *b = (double *)malloc((size_t)(N + 2) * sizeof(double));
    int64_t s;
    if (!a || !b) { free(a); free(b); return -1; }
    a[0] = bc_lo; a[N + 1] = bc_hi;
    memcpy(a + 1, u, (size_t)N * sizeof(double));
    for (s = 0; s < steps; ++s) {
        double *t;
        ge_ref_level_1d_var(a, b, N, rl, k, pmod(level0 + s, 2));
        t = a; a = b; b = t;
    }
    memcpy(u, a + 1, (size_t)N * sizeof(double));
    free(a); free(b);
    return 0;
}
