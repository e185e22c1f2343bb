"""Pins for the oracle's level with a source term and time-dependent boundary values
(oracle/ge_ref.c ge_ref_level_1d_src; reading R-N3) -- CPU only.
The paper has neither, so every pin is mathematical."""
import numpy as np
import pytest

import dense_ref as D


@pytest.mark.parametrize("k", [1, 2, 5])
@pytest.mark.parametrize("phase", [0, 1])
@pytest.mark.parametrize("n", [1, 2, 7, 16, 33])
def test_reduces_to_the_pinned_level_without_source_and_with_fixed_boundaries(oracle, k, phase, n):
    rng = np.random.default_rng(n + k)
    u = rng.uniform(-1, 1, n)
    for r in (0.5, 2.0, 7.0):
        a = oracle.level_1d(u, r, phase, 0.3, -0.7, k=k)
        b = oracle.level_1d_src(u, r, phase, (0.3, -0.7), (0.3, -0.7), None, k=k)
        c = oracle.level_1d_src(u, r, phase, (0.3, -0.7), (0.3, -0.7), np.zeros(n), k=k)
        np.testing.assert_array_equal(a, b)
        np.testing.assert_array_equal(a, c)


@pytest.mark.parametrize("k", [1, 2, 3])
@pytest.mark.parametrize("phase", [0, 1])
@pytest.mark.parametrize("n", [1, 2, 3, 6, 9, 16])
def test_brute_force_from_the_implicit_statement(oracle, k, phase, n):
    """Dense A^-1 (B old + c) assembled node by node, never touching Eqs (3),(4)."""
    rng = np.random.default_rng(100 * n + k)
    for r in (0.5, 1.0, 4.0, 25.0):
        u = rng.uniform(-1, 1, n)
        s = rng.uniform(-0.5, 0.5, n)
        bo, bn = tuple(rng.uniform(-1, 1, 2)), tuple(rng.uniform(-1, 1, 2))
        got = oracle.level_1d_src(u, r, phase, bo, bn, s, k=k)
        ref = D.level_1d_dense_src(u, r, k, phase, bo, bn, s)
        np.testing.assert_allclose(got, ref, rtol=0, atol=2e-13 * max(1.0, r))


@pytest.mark.parametrize("k", [1, 2, 16])
@pytest.mark.parametrize("n", [8, 31, 62])
def test_linear_in_space_and_time_is_reproduced_exactly(oracle, k, n):
    """u = a + b x + c t with f = c and boundaries a + c t, a + b + c t is an exact solution of every
    formula (second difference zero, time difference tau*c): any r, both phases, any k."""
    a, b, c = 0.4, -1.3, 2.5
    h = 1.0 / (n + 1)
    x = np.arange(1, n + 1) * h
    for r in (0.5, 3.0):
        tau = r * h * h
        u, t = a + b * x, 0.0
        for level in range(6):
            bo, bn = (a + c * t, a + b + c * t), (a + c * (t + tau), a + b + c * (t + tau))
            u = oracle.level_1d_src(u, r, level % 2, bo, bn, np.full(n, tau * c), k=k)
            t += tau
            np.testing.assert_allclose(u, a + b * x + c * t, rtol=0, atol=1e-13)


def _manufactured(oracle, n, r, t_end):
    """u = e^{-pi^2 t} sin(pi x) + x t^2 + (1 - x) sin t : f = u_t - u_xx of the last two terms."""
    h = 1.0 / (n + 1)
    x = np.arange(1, n + 1) * h
    tau = r * h * h
    steps = int(round(t_end / tau))
    steps += steps % 2
    exact = lambda t: np.exp(-np.pi ** 2 * t) * np.sin(np.pi * x) + x * t * t + (1 - x) * np.sin(t)
    f = lambda t: 2 * x * t + (1 - x) * np.cos(t)
    lo, hi = (lambda t: np.sin(t)), (lambda t: t * t)
    u, t = exact(0.0), 0.0
    for level in range(steps):
        u = oracle.level_1d_src(u, r, level % 2, (lo(t), hi(t)), (lo(t + tau), hi(t + tau)), tau * f(t + tau / 2))
        t += tau
    return float(np.abs(u - exact(t)).max())


def test_manufactured_solution_converges_at_second_order(oracle):
    errs = [_manufactured(oracle, n, 1.0, 0.1) for n in (31, 63, 127)]
    assert errs[0] / errs[1] > 3.5 and errs[1] / errs[2] > 3.5, errs
    assert errs[2] < 3e-4


def test_exact_rational_fixture(oracle):
    """tests/golden/p12_src_exact.txt: two levels with a source term and moving boundary values, exact rationals."""
    from fractions import Fraction as F
    from conftest import golden_lines
    for ln in golden_lines("p12_src_exact.txt"):
        head, lo, hi, u0, s1, s2, u1, u2 = [p.strip() for p in ln.split(";")]
        k, r = int(head.split()[0]), float(F(head.split()[1]))
        vec = lambda t: np.array([float(F(x)) for x in t.split()])
        lo, hi, u0, s1, s2, u1, u2 = map(vec, (lo, hi, u0, s1, s2, u1, u2))
        g1 = oracle.level_1d_src(u0, r, 0, (lo[0], hi[0]), (lo[1], hi[1]), s1, k=k)
        np.testing.assert_allclose(g1, u1, rtol=0, atol=1e-13)
        g2 = oracle.level_1d_src(g1, r, 1, (lo[1], hi[1]), (lo[2], hi[2]), s2, k=k)
        np.testing.assert_allclose(g2, u2, rtol=0, atol=1e-13)
