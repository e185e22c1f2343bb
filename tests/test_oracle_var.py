"""Pins for the oracle's level with VARIABLE DIFFUSIVITY (oracle/ge_ref.c ge_ref_level_1d_var; DESIGN.md reading
R-VAR) -- CPU only.  The paper's model problem has a constant coefficient
(PAPER.md:57-61), so every pin is mathematical: reduction to the pinned constant-r level, exact rationals and a
dense brute force from the implicit statement (a second derivation that never touches the pair's closed form),
invariants, stability of the two-level cycle, and convergence to an exact steady state."""
from fractions import Fraction

import numpy as np
import pytest

import dense_ref as D


@pytest.mark.parametrize("k", [1, 2, 5])
@pytest.mark.parametrize("phase", [0, 1])
@pytest.mark.parametrize("n", [1, 2, 3, 7, 16, 33])
def test_constant_coefficient_reduces_to_the_pinned_level(oracle, k, phase, n):
    """rl[j] = r for every link: Eqs (1)-(4) of the paper.  The two functions write the pair differently (four
    printed weights against (1+r) p + r q), so they agree to rounding, not bit for bit."""
    rng = np.random.default_rng(n + 10 * k)
    u = rng.uniform(-1, 1, n)
    for r in (0.5, 2.0, 7.0):
        a = oracle.level_1d(u, r, phase, 0.3, -0.7, k=k)
        b = oracle.level_1d_var(u, np.full(n + 1, r), phase, 0.3, -0.7, k=k)
        np.testing.assert_allclose(a, b, rtol=0, atol=4e-15 * max(1.0, r))


def test_exact_rational_worked_examples(oracle):
    """Small cases solved over the rationals from the implicit statement (dense_ref.system_1d_var), compared with
    the oracle's floating-point closed forms: every formula, truncated groups, k = 1 and 2, odd N."""
    cases = [
        (1, [1, 2, 3, 4], [1, 2, 3, 1, 2], 0, 0),
        (1, [4, 0, 0, 8, 2, 6], [Fraction(1, 2), 2, 1, 3, Fraction(3, 2), 2, 1], 1, 3),
        (1, [1, 2, 3, 4, 5, 6, 7], [2, 1, 3, 1, 2, 1, 3, 2], 0, 0),
        (2, [1, 2, 3, 4, 5, 6], [1, 2, 1, 3, 1, 2, 1], 0, 0),
        (2, [3, -1, 4, 1, -5, 9, 2], [2, 1, Fraction(1, 2), 3, 1, 2, 1, 4], -1, 2),
    ]
    for k, u0, rl, lo, hi in cases:
        u_exact = [Fraction(x) for x in u0]
        u_float = np.array(u0, dtype=np.float64)
        for level in range(4):
            u_exact = D.level_1d_var_exact(u_exact, rl, k, level % 2, lo, hi)
            u_float = oracle.level_1d_var(u_float, np.array([float(x) for x in rl]), level % 2, lo, hi, k=k)
            np.testing.assert_allclose(u_float, [float(x) for x in u_exact], rtol=0, atol=5e-13)
    # one value by hand: N = 2, phase 0, links (1, 2, 3), u0 = (1, 2), zero boundaries:
    # p = (1-1) 1 + 1*0 = 0, q = (1-3) 2 + 3*0 = -4, rm = 2: new_1 = (3*0 + 2*(-4))/5 = -8/5, new_2 = (2*0 + 3*(-4))/5 = -12/5
    got = oracle.level_1d_var(np.array([1.0, 2.0]), np.array([1.0, 2.0, 3.0]), 0)
    np.testing.assert_allclose(got, [-8 / 5, -12 / 5], rtol=0, atol=1e-15)


@pytest.mark.parametrize("k", [1, 2, 3])
@pytest.mark.parametrize("phase", [0, 1])
@pytest.mark.parametrize("n", [1, 2, 3, 6, 9, 16])
def test_brute_force_from_the_implicit_statement(oracle, k, phase, n):
    rng = np.random.default_rng(100 * n + k)
    for scale in (0.5, 4.0, 25.0):
        u = rng.uniform(-1, 1, n)
        rl = rng.uniform(0.1, 1.0, n + 1) * scale
        lo, hi = rng.uniform(-1, 1, 2)
        got = oracle.level_1d_var(u, rl, phase, lo, hi, k=k)
        ref = D.level_1d_var_dense(u, rl, k, phase, lo, hi)
        np.testing.assert_allclose(got, ref, rtol=0, atol=2e-13 * max(1.0, scale))


@pytest.mark.parametrize("k", [1, 2, 16])
def test_invariants(oracle, k):
    """(i) constants are fixed points whatever the links (every formula's weights sum to one); (ii) the discrete
    steady state -- equal flux rl[j] (u_{j+1} - u_j) through every link -- is a fixed point of every formula;
    (iii) mirror symmetry: reversing the rod, the links and the boundary values reverses the result when the
    pair pattern is mirror-symmetric ((N + 2) mod 2k == 0)."""
    rng = np.random.default_rng(k)
    n = 62
    rl = rng.uniform(0.3, 6.0, n + 1)
    for phase in (0, 1):
        c = oracle.level_1d_var(np.full(n, 0.7), rl, phase, 0.7, 0.7, k=k)
        np.testing.assert_allclose(c, 0.7, rtol=0, atol=1e-15)
        # steady state: u_{j+1} - u_j = F / rl[j]
        full = np.concatenate([[0.25], 0.25 + np.cumsum(1.3 / rl)])
        s = oracle.level_1d_var(full[1:-1], rl, phase, full[0], full[-1], k=k)
        np.testing.assert_allclose(s, full[1:-1], rtol=0, atol=2e-13)
        u = rng.uniform(-1, 1, n)
        a = oracle.level_1d_var(u, rl, phase, 0.2, -0.4, k=k)
        b = oracle.level_1d_var(u[::-1].copy(), rl[::-1].copy(), phase, -0.4, 0.2, k=k)
        np.testing.assert_allclose(a, b[::-1], rtol=0, atol=1e-14)


@pytest.mark.parametrize("k", [1, 2, 3])
@pytest.mark.parametrize("n", [6, 8, 15, 16])
def test_two_level_cycle_is_stable_for_any_positive_links(oracle, k, n):
    """rho(T1 T0) <= 1 with link numbers spread over two decades (up to 100); a single level is not stable."""
    rng = np.random.default_rng(7 * n + k)
    worst_single = 0.0
    for trial in range(4):
        rl = 10.0 ** rng.uniform(0.0, 2.0, n + 1)
        t0 = D.operator_1d_var(n, rl, k, 0)
        t1 = D.operator_1d_var(n, rl, k, 1)
        # the dense operators are the oracle's: column by column
        for j in range(n):
            e = np.zeros(n); e[j] = 1.0
            np.testing.assert_allclose(oracle.level_1d_var(e, rl, 0, k=k), t0[:, j], rtol=0, atol=1e-12)
        rho = np.abs(np.linalg.eigvals(t1 @ t0)).max()
        assert rho <= 1.0 + 1e-10, (k, n, rho)
        worst_single = max(worst_single, np.abs(np.linalg.eigvals(t0)).max())
    assert worst_single > 1.5          # so nobody "fixes" the test by looking at one level


def test_converges_to_the_steady_state_of_a_variable_coefficient(oracle):
    """a(x) = 1 + x, u(0) = 0, u(1) = 1: the steady state of u_t = (a u_x)_x is u = ln(1 + x) / ln 2.  With
    a_{j+1/2} = 1 + (j + 1/2) h the marched solution settles on the DISCRETE steady state, whose distance to the
    exact one falls like h^2 (midpoint rule)."""
    errs = []
    for n in (15, 31, 63):
        h = 1.0 / (n + 1)
        x = np.arange(1, n + 1) * h
        r = 1.0
        rl = r * (1.0 + (np.arange(n + 1) + 0.5) * h)
        u = oracle.run_1d_var(x.copy(), rl, 60 * (n + 1) ** 2 // 10 * 2, 0.0, 1.0)
        errs.append(np.abs(u - np.log1p(x) / np.log(2.0)).max())
    assert errs[0] / errs[1] > 3.5 and errs[1] / errs[2] > 3.5, errs
    assert errs[2] < 2e-5, errs


def test_run_equals_levels(oracle):
    rng = np.random.default_rng(3)
    n = 41
    u = rng.uniform(-1, 1, n); rl = rng.uniform(0.5, 5, n + 1)
    for k in (1, 4):
        a = u.copy()
        for lev in range(7):
            a = oracle.level_1d_var(a, rl, (lev + 1) % 2, 0.1, 0.9, k=k)
        b = oracle.run_1d_var(u, rl, 7, 0.1, 0.9, k=k, level0=1)
        np.testing.assert_array_equal(a, b)
