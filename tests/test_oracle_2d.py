"""Pins for the 2-D oracle (reading R-2D; PAPER.md defines no 2-D scheme,
PAPER.md:134, :228) -- CPU only.  SURVEY.md 8(c) P2, P4, P5, P6, P8, P9."""
from fractions import Fraction as F

import numpy as np
import pytest

from conftest import golden_lines
import dense_ref as D


@pytest.mark.parametrize("line", golden_lines("p9_2d_exact.txt"))
def test_p9_exact_rational_examples(oracle, line):
    head, u0, l1, l2 = [s.strip() for s in line.split(";")]
    n, r = head.split()
    n, r = int(n), F(r)
    sh = lambda s: [[F(t) for t in s.split()][j * n:(j + 1) * n] for j in range(n)]
    u0, l1, l2 = sh(u0), sh(l1), sh(l2)
    e1 = D.level_2d_exact(u0, r, 0)
    e2 = D.level_2d_exact(e1, r, 1)
    assert e1 == l1 and e2 == l2
    f = lambda m: np.array([[float(v) for v in row] for row in m])
    o1 = oracle.level_2d(f(u0), float(r), 0)
    o2 = oracle.level_2d(o1, float(r), 1)
    np.testing.assert_allclose(o1, f(l1), rtol=1e-14, atol=1e-15)
    np.testing.assert_allclose(o2, f(l2), rtol=1e-13, atol=1e-14)
    np.testing.assert_array_equal(oracle.run_2d(f(u0), float(r), 2), o2)


@pytest.mark.parametrize("nx,ny", [(1, 1), (2, 2), (3, 3), (4, 4), (5, 4), (4, 7), (6, 6), (7, 5), (8, 8), (1, 6), (6, 1)])
def test_p4_dense_brute_force_2d(oracle, nx, ny):
    rng = np.random.default_rng(10 * nx + ny)
    for phase in (0, 1):
        for r in (0.5, 1.0, 2.0, 10.0):
            u = rng.standard_normal((ny, nx))
            bc = tuple(rng.standard_normal(4))
            ref = D.level_2d_dense(u, r, phase, bc)
            got = oracle.level_2d(u, r, phase, bc)
            np.testing.assert_allclose(got, ref, rtol=0, atol=1e-13 * max(1.0, np.abs(ref).max()))


@pytest.mark.parametrize("n", [3, 4, 7, 8])
@pytest.mark.parametrize("phase", [0, 1])
def test_p2_constant_and_bilinear_fixed_points(oracle, n, phase):
    for r in (0.5, 2.0, 7.0):
        c = np.full((n, n), -0.75)
        np.testing.assert_allclose(oracle.level_2d(c, r, phase, (-0.75,) * 4), c, rtol=1e-13)
    # u = a + b*x (y-invariant, harmonic) with matching edges is a fixed point
    i = np.arange(0, n + 2, dtype=np.float64)
    lin = 1.0 + 0.25 * i
    u = np.tile(lin[1:-1], (n, 1))
    # edges y_lo / y_hi are not constant for this field, so check only via the dense statement instead:
    ref = D.level_2d_dense(u, 2.0, phase, (lin[0], lin[-1], 0.0, 0.0))
    np.testing.assert_allclose(oracle.level_2d(u, 2.0, phase, (lin[0], lin[-1], 0.0, 0.0)), ref, atol=1e-13)


def test_p2_symmetries(oracle):
    # even N: pattern is symmetric under x -> 1-x, y -> 1-y and transpose
    rng = np.random.default_rng(21)
    n = 8
    q = rng.standard_normal((n // 2, n // 2))
    u = np.block([[q, q[:, ::-1]], [q[::-1, :], q[::-1, ::-1]]])
    out = oracle.run_2d(u, 2.0, 6)
    np.testing.assert_allclose(out, out[:, ::-1], atol=1e-13)
    np.testing.assert_allclose(out, out[::-1, :], atol=1e-13)
    v = rng.standard_normal((n, n))
    np.testing.assert_allclose(oracle.run_2d(v.T.copy(), 3.0, 5), oracle.run_2d(v, 3.0, 5).T, atol=1e-13)


def _rho(M):
    return np.abs(np.linalg.eigvals(M)).max()


def _ops(oracle, n, r):
    eye = np.eye(n * n)
    T0 = np.stack([oracle.level_2d(e.reshape(n, n), r, 0).ravel() for e in eye], axis=1)
    T1 = np.stack([oracle.level_2d(e.reshape(n, n), r, 1).ravel() for e in eye], axis=1)
    return T0, T1


@pytest.mark.parametrize("n", [4, 6, 7, 8])
def test_p5_cycle_spectral_radius_le_one_2d(oracle, n):
    for r in (0.5, 1, 2, 10, 100):
        T0, T1 = _ops(oracle, n, r)
        assert _rho(T1 @ T0) <= 1.0 + 1e-12
        np.testing.assert_allclose(T0, D.operator_2d(n, n, r, 0), atol=1e-13)
        np.testing.assert_allclose(T1, D.operator_2d(n, n, r, 1), atol=1e-13)


def test_p5_golden_spectral_radii_2d(oracle):
    for ln in golden_lines("p5_spectral_radius.txt"):
        dim, n, k, r, rc, rs = ln.split()
        if dim != "2":
            continue
        T0, T1 = _ops(oracle, int(n), float(r))
        assert abs(_rho(T1 @ T0) - float(rc)) < 2e-6


def test_p5_axis_shift_would_be_caught(oracle):
    # without the diagonal alternation (phase 0 twice) the scheme is unstable at r = 2
    T0, _ = _ops(oracle, 6, 2.0)
    assert _rho(T0 @ T0) > 2.0


def test_p6_convergence_golden_2d(oracle):
    vals = {}
    for ln in golden_lines("p6_p7_convergence.txt"):
        f = ln.split()
        if f[0] == "maxerr" and f[1] == "2":
            n, r, t, v = int(f[2]), float(f[4]), float(f[5]), float(f[6])
            h = 1.0 / (n + 1)
            tau = r * h * h
            levels = 2 * int(round(t / tau / 2))
            x = np.arange(1, n + 1) * h
            s = np.outer(np.sin(np.pi * x), np.sin(np.pi * x))
            u = oracle.run_2d(s, r, levels)
            e = np.abs(u - np.exp(-2 * np.pi ** 2 * levels * tau) * s).max()
            vals[n] = e
            assert abs(e - v) < 8e-3 * v, (n, e, v)
    assert 3.4 < vals[16] / vals[32] < 4.2 and 3.4 < vals[32] / vals[64] < 4.2


def test_p8_y_invariant_data_reduce_to_1d_pairs(oracle):
    # rows far from the y-edges of y-invariant data follow the 1-D Eqs (3)/(4) for one level
    rng = np.random.default_rng(17)
    nx, ny, r = 12, 10, 1.5
    row = rng.standard_normal(nx)
    u = np.tile(row, (ny, 1))
    for phase in (0, 1):
        out = oracle.level_2d(u, r, phase, (0.3, -0.2, 0.0, 0.0))
        ref = oracle.level_1d(row, r, phase, 0.3, -0.2)
        for j in range(2, ny - 2):
            np.testing.assert_allclose(out[j], ref, rtol=1e-13, atol=1e-14)
