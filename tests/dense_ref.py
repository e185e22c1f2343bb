"""Second derivation of one GE level, used only by the oracle pin tests (P1, P4).

It never touches the closed forms (3)/(4) or the 4x4 inverse: every node gets
its *implicit* statement
    (1 + r*n_new) new_i - r * sum_{new-level nbrs} new_j
        = (1 - r*n_old) old_i + r * sum_{old-level nbrs} old_j
where the rule table (R-1D / R-2D) only decides which
neighbours are taken at the new level, and the system A new = B old + c is
solved densely (numpy, or exact Fractions).  Boundary nodes are known at both
levels and go to the constant vector c.
"""
from fractions import Fraction

import numpy as np


def classes_1d(n, k, phase):
    """'new-level neighbour' of every interior node 1..n: -1 (left), +1 (right)."""
    side = {}
    for i in range(1, n + 1):
        c = (i - phase * k) % (2 * k)
        if c == 2 * k - 1:      # left member of a pair: partner i+1 at the new level  (Eq 2 at i)
            side[i] = +1
        elif c == 0:            # right member: partner i-1 at the new level           (Eq 1 at i)
            side[i] = -1
        elif 1 <= c <= k - 1:   # Saul'yev A: left neighbour new
            side[i] = -1
        else:                   # Saul'yev B: right neighbour new
            side[i] = +1
    return side


def system_1d(n, r, k, phase, bc_lo, bc_hi, num=float):
    """Return (A, B, c) with A new = B old + c over interior nodes 1..n (index i-1)."""
    zero, one = num(0), num(1)
    A = [[zero] * n for _ in range(n)]
    B = [[zero] * n for _ in range(n)]
    c = [zero] * n
    bval = {0: num(bc_lo), n + 1: num(bc_hi)}
    side = classes_1d(n, k, phase)
    for i in range(1, n + 1):
        A[i - 1][i - 1] = one + r
        B[i - 1][i - 1] = one - r
        jn, jo = i + side[i], i - side[i]
        if jn in bval:
            c[i - 1] += r * bval[jn]
        else:
            A[i - 1][jn - 1] -= r
        if jo in bval:
            c[i - 1] += r * bval[jo]
        else:
            B[i - 1][jo - 1] += r
    return A, B, c


def level_1d_dense_src(u, r, k, phase, bc_old, bc_new, s=None):
    """Implicit statement with a source term and moving boundary values (reading R-N3): a boundary
    neighbour taken at the new level contributes its NEW value, one taken at the old level its OLD value."""
    n = len(u)
    r = float(r)
    A = np.zeros((n, n)); B = np.zeros((n, n)); c = np.zeros(n)
    side = classes_1d(n, k, phase)
    old_b = {0: bc_old[0], n + 1: bc_old[1]}
    new_b = {0: bc_new[0], n + 1: bc_new[1]}
    for i in range(1, n + 1):
        A[i - 1, i - 1] = 1 + r
        B[i - 1, i - 1] = 1 - r
        jn, jo = i + side[i], i - side[i]
        if jn in new_b:
            c[i - 1] += r * new_b[jn]
        else:
            A[i - 1, jn - 1] -= r
        if jo in old_b:
            c[i - 1] += r * old_b[jo]
        else:
            B[i - 1, jo - 1] += r
    if s is not None:
        c = c + np.asarray(s, dtype=np.float64)
    return np.linalg.solve(A, B @ np.asarray(u, dtype=np.float64) + c)


def system_1d_var(n, rl, k, phase, bc_lo, bc_hi, num=float):
    """Variable diffusivity (reading R-VAR): rl[j] belongs to the link between nodes j and j+1.  Node by node:
    (1 + r_new) new_i - r_new new_{jn} = (1 - r_old) old_i + r_old old_{jo}, the rule table only deciding which
    neighbour jn is taken at the new level.  Returns (A, B, c) with A new = B old + c."""
    zero, one = num(0), num(1)
    A = [[zero] * n for _ in range(n)]
    B = [[zero] * n for _ in range(n)]
    c = [zero] * n
    bval = {0: num(bc_lo), n + 1: num(bc_hi)}
    side = classes_1d(n, k, phase)
    for i in range(1, n + 1):
        jn, jo = i + side[i], i - side[i]
        rn, ro = num(rl[min(i, jn)]), num(rl[min(i, jo)])
        A[i - 1][i - 1] = one + rn
        B[i - 1][i - 1] = one - ro
        if jn in bval:
            c[i - 1] += rn * bval[jn]
        else:
            A[i - 1][jn - 1] -= rn
        if jo in bval:
            c[i - 1] += ro * bval[jo]
        else:
            B[i - 1][jo - 1] += ro
    return A, B, c


def level_1d_var_exact(u, rl, k, phase, bc_lo=0, bc_hi=0):
    n = len(u)
    A, B, c = system_1d_var(n, [Fraction(x) for x in rl], k, phase, bc_lo, bc_hi, num=Fraction)
    rhs = [sum(B[i][j] * Fraction(u[j]) for j in range(n)) + c[i] for i in range(n)]
    return solve_exact(A, rhs)


def level_1d_var_dense(u, rl, k, phase, bc_lo=0.0, bc_hi=0.0):
    n = len(u)
    A, B, c = system_1d_var(n, [float(x) for x in rl], k, phase, bc_lo, bc_hi)
    return np.linalg.solve(np.array(A), np.array(B) @ np.asarray(u, dtype=np.float64) + np.array(c))


def operator_1d_var(n, rl, k, phase):
    A, B, _ = system_1d_var(n, [float(x) for x in rl], k, phase, 0.0, 0.0)
    return np.linalg.solve(np.array(A), np.array(B))


def solve_exact(A, b):
    """Gaussian elimination over Fractions."""
    n = len(A)
    M = [row[:] + [b[i]] for i, row in enumerate(A)]
    for col in range(n):
        piv = next(rw for rw in range(col, n) if M[rw][col] != 0)
        M[col], M[piv] = M[piv], M[col]
        inv = Fraction(1) / M[col][col]
        M[col] = [v * inv for v in M[col]]
        for rw in range(n):
            if rw != col and M[rw][col] != 0:
                f = M[rw][col]
                M[rw] = [a - f * p for a, p in zip(M[rw], M[col])]
    return [M[i][n] for i in range(n)]


def level_1d_exact(u, r, k, phase, bc_lo=0, bc_hi=0):
    n = len(u)
    r = Fraction(r)
    A, B, c = system_1d(n, r, k, phase, bc_lo, bc_hi, num=Fraction)
    rhs = [sum(B[i][j] * Fraction(u[j]) for j in range(n)) + c[i] for i in range(n)]
    return solve_exact(A, rhs)


def level_1d_dense(u, r, k, phase, bc_lo=0.0, bc_hi=0.0):
    n = len(u)
    A, B, c = system_1d(n, float(r), k, phase, bc_lo, bc_hi)
    A, B, c = np.array(A), np.array(B), np.array(c)
    return np.linalg.solve(A, B @ np.asarray(u, dtype=np.float64) + c)


def operator_1d(n, r, k, phase):
    """Dense one-level operator for zero boundary values: inv(A) B."""
    A, B, _ = system_1d(n, float(r), k, phase, 0.0, 0.0)
    return np.linalg.solve(np.array(A), np.array(B))


def system_2d(nx, ny, r, phase, bc, num=float):
    """2-D: in-group neighbours at the new level, out-of-group at the old level.
    Unknown index (j-1)*nx + (i-1) for node (i,j); bc = (x_lo, x_hi, y_lo, y_hi)."""
    zero, one = num(0), num(1)
    n = nx * ny
    A = [[zero] * n for _ in range(n)]
    B = [[zero] * n for _ in range(n)]
    c = [zero] * n

    def group(i, j):
        return ((i - 1 + phase) // 2 if phase == 0 else (i // 2)), ((j - 1 + phase) // 2 if phase == 0 else (j // 2))

    def bvalue(i, j):
        if i == 0:
            return num(bc[0])
        if i == nx + 1:
            return num(bc[1])
        if j == 0:
            return num(bc[2])
        if j == ny + 1:
            return num(bc[3])
        return None

    for j in range(1, ny + 1):
        for i in range(1, nx + 1):
            p = (j - 1) * nx + (i - 1)
            A[p][p] = one + 2 * r
            B[p][p] = one - 2 * r
            for (qi, qj) in ((i - 1, j), (i + 1, j), (i, j - 1), (i, j + 1)):
                same = group(qi, qj) == group(i, j)
                bv = bvalue(qi, qj)
                if bv is not None:
                    c[p] += r * bv
                elif same:
                    A[p][(qj - 1) * nx + (qi - 1)] -= r
                else:
                    B[p][(qj - 1) * nx + (qi - 1)] += r
    return A, B, c


def level_2d_exact(u, r, phase, bc=(0, 0, 0, 0)):
    ny, nx = len(u), len(u[0])
    r = Fraction(r)
    A, B, c = system_2d(nx, ny, r, phase, bc, num=Fraction)
    flat = [Fraction(v) for row in u for v in row]
    n = nx * ny
    rhs = [sum(B[i][j] * flat[j] for j in range(n) if B[i][j] != 0) + c[i] for i in range(n)]
    sol = solve_exact(A, rhs)
    return [sol[j * nx:(j + 1) * nx] for j in range(ny)]


def level_2d_dense(u, r, phase, bc=(0.0, 0.0, 0.0, 0.0)):
    u = np.asarray(u, dtype=np.float64)
    ny, nx = u.shape
    A, B, c = system_2d(nx, ny, float(r), phase, bc)
    return np.linalg.solve(np.array(A), np.array(B) @ u.ravel() + np.array(c)).reshape(ny, nx)


def operator_2d(nx, ny, r, phase):
    A, B, _ = system_2d(nx, ny, float(r), phase, (0.0, 0.0, 0.0, 0.0))
    return np.linalg.solve(np.array(A), np.array(B))


def system_3d(nx, ny, nz, r, phase, bc, num=float):
    """3-D (reading R-3D): in-group neighbours at the new level, out-of-group at the old level.
    Unknown index ((k-1)*ny + (j-1))*nx + (i-1); bc = (x_lo, x_hi, y_lo, y_hi, z_lo, z_hi)."""
    zero, one = num(0), num(1)
    n = nx * ny * nz
    A = [[zero] * n for _ in range(n)]
    B = [[zero] * n for _ in range(n)]
    c = [zero] * n
    dims = (nx, ny, nz)

    def gid(p):
        return tuple(((q - 1) // 2 if phase == 0 else q // 2) for q in p)

    def bvalue(p):
        for ax in range(3):
            if p[ax] == 0:
                return num(bc[2 * ax])
            if p[ax] == dims[ax] + 1:
                return num(bc[2 * ax + 1])
        return None

    def index(p):
        return ((p[2] - 1) * ny + (p[1] - 1)) * nx + (p[0] - 1)

    for k in range(1, nz + 1):
        for j in range(1, ny + 1):
            for i in range(1, nx + 1):
                p = (i, j, k)
                row = index(p)
                A[row][row] = one + 3 * r
                B[row][row] = one - 3 * r
                for ax in range(3):
                    for d in (-1, 1):
                        q = list(p); q[ax] += d; q = tuple(q)
                        bv = bvalue(q)
                        if bv is not None:
                            c[row] += r * bv
                        elif gid(q) == gid(p):
                            A[row][index(q)] -= r
                        else:
                            B[row][index(q)] += r
    return A, B, c


def level_3d_dense(u, r, phase, bc=(0.0,) * 6):
    u = np.asarray(u, dtype=np.float64)
    nz, ny, nx = u.shape
    A, B, c = system_3d(nx, ny, nz, float(r), phase, bc)
    return np.linalg.solve(np.array(A), np.array(B) @ u.ravel() + np.array(c)).reshape(nz, ny, nx)


def operator_3d(nx, ny, nz, r, phase):
    A, B, _ = system_3d(nx, ny, nz, float(r), phase, (0.0,) * 6)
    return np.linalg.solve(np.array(A), np.array(B))
