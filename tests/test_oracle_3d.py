"""Pins for the 3-D oracle (oracle/ge_ref.c ge_ref_level_3d; reading R-3D, SURVEY.md 8(f)
NEXT-4) -- CPU only.  PAPER.md defines no 3-D scheme (PAPER.md:134, :228 only claim the extension), so
the reading is pinned by mathematics: invariants, dense brute force from the implicit statement,
exact rationals, spectral radius of the two-level cycle, convergence to the closed form."""
from fractions import Fraction as F

import numpy as np
import pytest

import dense_ref as D


@pytest.mark.parametrize("phase", [0, 1])
@pytest.mark.parametrize("shape", [(1, 1, 1), (2, 2, 2), (3, 2, 4), (4, 4, 4), (5, 3, 2)])
def test_constants_and_linear_data_are_fixed_points(oracle, phase, shape):
    nz, ny, nx = shape
    for r in (0.5, 2.0, 9.0):
        c = np.full(shape, 1.75)
        np.testing.assert_allclose(oracle.level_3d(c, r, phase, (1.75,) * 6), c, rtol=1e-14)
        k, j, i = np.meshgrid(np.arange(nz + 2), np.arange(ny + 2), np.arange(nx + 2), indexing="ij")
        lin = 0.5 - 0.125 * i + 0.25 * j + 0.0625 * k        # second differences vanish in every axis
        new = oracle.level_3d_padded(lin, r, phase)
        np.testing.assert_allclose(new[1:-1, 1:-1, 1:-1], lin[1:-1, 1:-1, 1:-1], rtol=0, atol=1e-13)


@pytest.mark.parametrize("phase", [0, 1])
@pytest.mark.parametrize("shape", [(1, 1, 1), (2, 2, 2), (2, 3, 1), (3, 3, 3), (4, 4, 4), (4, 2, 5), (3, 5, 4)])
def test_brute_force_from_the_implicit_statement(oracle, phase, shape):
    """Global dense A^-1 (B old + c), assembled node by node; the oracle solves group by group."""
    rng = np.random.default_rng(sum(shape) + phase)
    for r in (0.5, 1.0, 4.0, 30.0):
        u = rng.uniform(-1, 1, shape)
        bc = tuple(rng.uniform(-1, 1, 6))
        got = oracle.level_3d(u, r, phase, bc)
        ref = D.level_3d_dense(u, r, phase, bc)
        np.testing.assert_allclose(got, ref, rtol=0, atol=3e-13 * max(1.0, r))


def test_exact_rational_full_group():
    """N = 2, phase 0: one full 2x2x2 group, zero boundary values, r = 1: (1+3r) I - r Q3 solved in
    exact rationals; by symmetry u0 = 1 everywhere gives R = 1 - 3r = -2 and new = -2 / (1+3r-3r) = -2."""
    A, B, c = D.system_3d(2, 2, 2, F(1), 0, (0,) * 6, num=F)
    rhs = [sum(B[i][j] for j in range(8)) + c[i] for i in range(8)]
    sol = D.solve_exact(A, rhs)
    assert all(v == F(-2) for v in sol)
    # a single hot corner: eigen-decomposition of the cube graph gives the exact weights
    rhs = [B[i][0] for i in range(8)]
    sol = D.solve_exact(A, rhs)
    lam = {0: F(1), 1: F(3), 2: F(5), 3: F(7)}           # 1 + 3r - r*(3 - 2*popcount) at r = 1
    for d in range(8):
        w = sum(F((-1) ** bin(d & m).count("1")) / lam[bin(m).count("1")] for m in range(8)) / 8
        assert sol[d] == (1 - 3) * w                      # B[0][0] = 1 - 3r = -2


def test_exact_rational_matches_oracle(oracle):
    u = np.arange(1, 9, dtype=np.float64).reshape(2, 2, 2)
    A, B, c = D.system_3d(2, 2, 2, F(2), 0, (1, 0, 0, 3, 0, 0), num=F)
    flat = [F(int(v)) for v in u.ravel()]
    rhs = [sum(B[i][j] * flat[j] for j in range(8)) + c[i] for i in range(8)]
    sol = np.array([float(v) for v in D.solve_exact(A, rhs)]).reshape(2, 2, 2)
    np.testing.assert_allclose(oracle.level_3d(u, 2.0, 0, (1, 0, 0, 3, 0, 0)), sol, rtol=0, atol=1e-13)
    # phase 1 on N = 2: eight single-member corner groups
    A, B, c = D.system_3d(2, 2, 2, F(2), 1, (1, 0, 0, 3, 0, 0), num=F)
    rhs = [sum(B[i][j] * flat[j] for j in range(8)) + c[i] for i in range(8)]
    sol = np.array([float(v) for v in D.solve_exact(A, rhs)]).reshape(2, 2, 2)
    np.testing.assert_allclose(oracle.level_3d(u, 2.0, 1, (1, 0, 0, 3, 0, 0)), sol, rtol=0, atol=1e-13)


@pytest.mark.parametrize("n", [3, 4])
def test_two_level_cycle_is_unconditionally_stable(n):
    for r in (0.5, 1.0, 2.0, 10.0, 100.0):
        T0, T1 = D.operator_3d(n, n, n, r, 0), D.operator_3d(n, n, n, r, 1)
        rho = max(abs(np.linalg.eigvals(T1 @ T0)))
        assert rho <= 1.0 + 1e-10, (n, r, rho)
    # a single level is NOT stable beyond r ~ 1: nobody should "fix" the alternation
    assert max(abs(np.linalg.eigvals(D.operator_3d(4, 4, 4, 4.0, 0)))) > 1.0


def test_convergence_to_the_closed_form(oracle):
    """u = e^{-3 pi^2 t} sin(pi x) sin(pi y) sin(pi z), zero boundary values, r = 1, t ~ 0.03."""
    errs = []
    for n in (7, 15, 31):
        h = 1.0 / (n + 1)
        x = np.arange(1, n + 1) * h
        u0 = np.sin(np.pi * x)[None, None, :] * np.sin(np.pi * x)[None, :, None] * np.sin(np.pi * x)[:, None, None]
        steps = int(round(0.03 / (h * h))); steps += steps % 2
        t = steps * h * h
        u = oracle.run_3d(u0, 1.0, steps)
        errs.append(float(np.abs(u - np.exp(-3 * np.pi ** 2 * t) * u0).max()))
    assert errs[0] / errs[1] > 3.0 and errs[1] / errs[2] > 3.3, errs


def test_exact_rational_fixture(oracle):
    """tests/golden/p11_3d_exact.txt: two levels in exact rationals from the implicit statement."""
    from conftest import golden_lines
    for ln in golden_lines("p11_3d_exact.txt"):
        head, bc, u0, u1, u2 = [p.strip() for p in ln.split(";")]
        n, r = int(head.split()[0]), float(F(head.split()[1]))
        bc = tuple(float(F(t)) for t in bc.split())
        a0 = np.array([float(F(t)) for t in u0.split()]).reshape(n, n, n)
        a1 = np.array([float(F(t)) for t in u1.split()]).reshape(n, n, n)
        a2 = np.array([float(F(t)) for t in u2.split()]).reshape(n, n, n)
        g1 = oracle.level_3d(a0, r, 0, bc)
        np.testing.assert_allclose(g1, a1, rtol=0, atol=1e-12)
        np.testing.assert_allclose(oracle.level_3d(g1, r, 1, bc), a2, rtol=0, atol=1e-12)
        np.testing.assert_allclose(oracle.run_3d(a0, r, 2, bc), a2, rtol=0, atol=1e-12)


def _walsh_group(R, r, axes):
    """Closed form of one group in exact rationals, a derivation that never assembles a matrix: the group's block
    is (1+3r) I - r (sum of the partner swaps along the group's `axes`), the swaps commute, their common
    eigenvectors are the Walsh functions h_m[d] = (-1)^popcount(d & m) with eigenvalue
    1 + 3r - r (number of axes) + 2 r popcount(m); new = sum_m h_m <h_m, b> / (2^axes lambda_m)."""
    n = 1 << axes
    out = []
    for d in range(n):
        acc = F(0)
        for m in range(n):
            lam = 1 + 3 * r - r * axes + 2 * r * bin(m).count("1")
            coef = sum(F((-1) ** bin(e & m).count("1")) * R[e] for e in range(n))
            acc += F((-1) ** bin(d & m).count("1")) * coef / (n * lam)
        out.append(acc)
    return out


@pytest.mark.parametrize("r", [F(1, 2), F(2), F(7)])
def test_walsh_closed_form_in_exact_rationals(oracle, r):
    """The oracle eliminates every group's block numerically; here the same level comes from the Walsh / Kronecker
    closed form in exact rationals (a second derivation: no matrix, no elimination) -- a full 2x2x2 group whose
    out-of-group neighbours are all boundary values, a full group with interior out-of-group neighbours, and the
    groups cut by one face (a 2x2 square: eigenvalues 1+r, 1+3r, 1+3r, 1+5r -- the form the CUDA kernels use,
    csrc/ge_level3d.cuh cut4_solve), by an edge (a pair: 1+2r, 1+4r) and by a corner (one node: 1+3r)."""
    rng = np.random.default_rng(int(r * 2))
    bc = (F(3), F(-1), F(2), F(5), F(-4), F(1))                      # x_lo, x_hi, y_lo, y_hi, z_lo, z_hi
    bcf = tuple(float(v) for v in bc)
    for phase, shape in ((0, (2, 2, 2)), (0, (1, 2, 2)), (1, (3, 3, 3)), (1, (2, 3, 3)), (0, (3, 3, 3))):
        nz, ny, nx = shape
        u = rng.integers(-9, 10, size=shape)
        val = lambda x, y, z: (bc[0] if x < 0 else bc[1] if x >= nx else bc[2] if y < 0 else bc[3] if y >= ny
                               else bc[4] if z < 0 else bc[5] if z >= nz else F(int(u[z, y, x])))
        expect = np.zeros(shape)
        first = lambda n: range(-phase, n, 2)                        # anchors -phase, 2 - phase, ... <= n - 1
        for gz in first(nz):
            for gy in first(ny):
                for gx in first(nx):
                    # the axes along which both nodes of the group are inside, and its interior members
                    inside = [[g + t for t in (0, 1) if 0 <= g + t < n] for g, n in ((gx, nx), (gy, ny), (gz, nz))]
                    full = [a for a in range(3) if len(inside[a]) == 2]
                    members = [(x, y, z) for z in inside[2] for y in inside[1] for x in inside[0]]   # x fastest
                    b = []
                    for (x, y, z) in members:
                        o = val(x, y, z)
                        s = F(0)
                        for a, (p, g) in enumerate(((x, gx), (y, gy), (z, gz))):
                            q = [x, y, z]
                            q[a] = p - 1 if p == g else p + 1        # the neighbour OUTSIDE the group along axis a
                            s += val(*q) - o
                        rhs = o + r * s                              # (1 - 3r) old + r (three out-of-group neighbours)
                        for a in range(3):                           # an in-group partner that is a boundary node: new level
                            if a not in full:
                                q = [x, y, z]
                                q[a] = -1 if [gx, gy, gz][a] < 0 else [nx, ny, nz][a]
                                rhs += r * val(*q)
                        b.append(rhs)
                    new = _walsh_group(b, r, len(full))
                    for (x, y, z), v in zip(members, new):
                        expect[z, y, x] = float(v)
        got = oracle.level_3d(u.astype(np.float64), float(r), phase, bcf)
        np.testing.assert_allclose(got, expect, rtol=0, atol=2e-13 * max(1.0, float(r)), err_msg=str((phase, shape)))
