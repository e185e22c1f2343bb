"""Pins for the 1-D oracle (oracle/ge_ref.c) -- CPU only.  SURVEY.md 8(c) P1-P8, P10.

PAPER.md prints no worked values, so every pin is mathematical: exact rationals
from the implicit statement, invariants, dense brute force, spectral radii,
convergence to the closed form named in BASELINE.json's north_star.
"""
from fractions import Fraction as F

import numpy as np
import pytest

from conftest import golden_lines
import dense_ref as D


def _fr(tok):
    return [F(t) for t in tok.split()]


# ---- P1: Eqs (3),(4) are the 2x2 solve of Eq (2)@i coupled with Eq (1)@i+1 ----
@pytest.mark.parametrize("r", [F(1, 2), F(1), F(2), F(7, 3), F(100)])
def test_p1_pair_weights_are_the_2x2_solve(oracle, r):
    # exact: (1+r)x - r y = (1-r) b + r a ;  -r x + (1+r) y = (1-r) c + r d   for old values a,b,c,d
    for col in range(4):
        old = [F(0)] * 4
        old[col] = F(1)
        a, b, c, d = old
        x, y = D.solve_exact([[1 + r, -r], [-r, 1 + r]], [(1 - r) * b + r * a, (1 - r) * c + r * d])
        w3 = [(r + r * r), (1 - r * r), (r - r * r), r * r]           # Eq (3) bracket
        w4 = [r * r, (r - r * r), (1 - r * r), (r + r * r)]           # Eq (4) bracket
        assert x == w3[col] / (1 + 2 * r) and y == w4[col] / (1 + 2 * r)
        # and NOT the garbled printed prefactor 1/(3(1+2r)) (reading R-A1)
        assert sum(w3) == 1 + 2 * r
    # oracle on a rod long enough that the pair (3,4) is interior: phase 0, k=1
    for col in range(2, 6):
        u = np.zeros(8)
        u[col - 1] = 1.0                                              # node `col`
        new = oracle.level_1d(u, float(r), 0)
        w3 = [(r + r * r), (1 - r * r), (r - r * r), r * r]
        w4 = [r * r, (r - r * r), (1 - r * r), (r + r * r)]
        np.testing.assert_allclose(new[2], float(w3[col - 2] / (1 + 2 * r)), rtol=1e-14, atol=1e-300)
        np.testing.assert_allclose(new[3], float(w4[col - 2] / (1 + 2 * r)), rtol=1e-14, atol=1e-300)


# ---- P2: invariants ----
@pytest.mark.parametrize("k", [1, 2, 3, 16])
@pytest.mark.parametrize("phase", [0, 1])
@pytest.mark.parametrize("n", [1, 2, 5, 8, 37, 62])
def test_p2_constants_and_linear_data_are_fixed_points(oracle, k, phase, n):
    for r in (0.5, 2.0, 9.0):
        c = np.full(n, 1.75)
        np.testing.assert_allclose(oracle.level_1d(c, r, phase, 1.75, 1.75, k=k), c, rtol=1e-14)
        i = np.arange(0, n + 2, dtype=np.float64)
        lin = 0.5 - 0.125 * i
        np.testing.assert_allclose(oracle.level_1d(lin[1:-1], r, phase, lin[0], lin[-1], k=k),
                                   lin[1:-1], rtol=1e-13, atol=1e-14)


@pytest.mark.parametrize("n,k", [(8, 1), (64, 1), (30, 2), (62, 16), (10, 3)])
def test_p2_mirror_symmetry(oracle, n, k):
    # even N at k=1, (N+2) mod 2k == 0 at k>=2: the pattern is mirror symmetric, so symmetric data stay symmetric
    rng = np.random.default_rng(7)
    half = rng.standard_normal(n // 2)
    u = np.concatenate([half, half[::-1]])
    out = oracle.run_1d(u, 3.0, 6, 0.25, 0.25, k=k)
    np.testing.assert_allclose(out, out[::-1], rtol=1e-12, atol=1e-14)
    # and an asymmetric pattern breaks the test's sensitivity check: odd N at k=1 is not symmetric per level
    one = oracle.level_1d(np.ones(7), 3.0, 0, 0.0, 0.0, k=1)
    assert abs(one[0] - one[-1]) > 1e-3


# ---- P3: exact-rational worked examples (tests/golden/p3_1d_exact.txt) ----
@pytest.mark.parametrize("line", golden_lines("p3_1d_exact.txt"))
def test_p3_exact_rational_examples(oracle, line):
    head, u0, l1, l2 = [s.strip() for s in line.split(";")]
    k, r, lo, hi = head.split()
    k, r, lo, hi = int(k), F(r), F(lo), F(hi)
    u0, l1, l2 = _fr(u0), _fr(l1), _fr(l2)
    # the fixture itself is re-derived exactly from the implicit statement (second derivation)
    e1 = D.level_1d_exact(u0, r, k, 0, lo, hi)
    e2 = D.level_1d_exact(e1, r, k, 1, lo, hi)
    assert e1 == l1 and e2 == l2
    o1 = oracle.level_1d([float(v) for v in u0], float(r), 0, float(lo), float(hi), k=k)
    o2 = oracle.level_1d(o1, float(r), 1, float(lo), float(hi), k=k)
    np.testing.assert_allclose(o1, [float(v) for v in l1], rtol=1e-14, atol=1e-15)
    np.testing.assert_allclose(o2, [float(v) for v in l2], rtol=1e-14, atol=2e-15)
    # run_1d (two levels from level 0) agrees with two level_1d calls
    np.testing.assert_array_equal(oracle.run_1d([float(v) for v in u0], float(r), 2, float(lo), float(hi), k=k), o2)


# ---- P4: brute force on tiny grids against the dense implicit statement ----
@pytest.mark.parametrize("k", [1, 2, 3, 5])
@pytest.mark.parametrize("n", [1, 2, 3, 6, 8, 15, 16])
def test_p4_dense_brute_force(oracle, n, k):
    rng = np.random.default_rng(100 * n + k)
    for phase in (0, 1):
        for r in (0.5, 1.0, 4.0, 10.0):
            u = rng.standard_normal(n)
            lo, hi = rng.standard_normal(2)
            ref = D.level_1d_dense(u, r, k, phase, lo, hi)
            got = oracle.level_1d(u, r, phase, lo, hi, k=k)
            np.testing.assert_allclose(got, ref, rtol=0, atol=1e-13 * max(1.0, np.abs(ref).max()))
            # (a) operator built column by column from the oracle acts like the oracle
            T = np.stack([oracle.level_1d(e, r, phase, 0.0, 0.0, k=k) for e in np.eye(n)], axis=1)
            np.testing.assert_allclose(T @ u, oracle.level_1d(u, r, phase, 0.0, 0.0, k=k), atol=1e-12)
            np.testing.assert_allclose(T, D.operator_1d(n, r, k, phase), atol=1e-13)


# ---- P5: unconditional stability of the two-level cycle ----
def _rho(M):
    return np.abs(np.linalg.eigvals(M)).max()


@pytest.mark.parametrize("k", [1, 2, 3])
@pytest.mark.parametrize("n", [6, 8, 15, 16])
def test_p5_cycle_spectral_radius_le_one(oracle, n, k):
    for r in (0.5, 1, 2, 4, 10, 100):
        T0 = np.stack([oracle.level_1d(e, r, 0, k=k) for e in np.eye(n)], axis=1)
        T1 = np.stack([oracle.level_1d(e, r, 1, k=k) for e in np.eye(n)], axis=1)
        assert _rho(T1 @ T0) <= 1.0 + 1e-12


def test_p5_golden_spectral_radii(oracle):
    for ln in golden_lines("p5_spectral_radius.txt"):
        dim, n, k, r, rc, rs = ln.split()
        if dim != "1":
            continue
        n, k, r = int(n), int(k), float(r)
        T0 = np.stack([oracle.level_1d(e, r, 0, k=k) for e in np.eye(n)], axis=1)
        T1 = np.stack([oracle.level_1d(e, r, 1, k=k) for e in np.eye(n)], axis=1)
        assert abs(_rho(T1 @ T0) - float(rc)) < 2e-6
        # a single level is NOT contractive for r > 1 (reading R-A13): nobody should "fix" this
        assert abs(_rho(T0) - float(rs)) < 6e-4 * float(rs) + 6e-4


def test_p5_wrong_alternation_would_be_caught(oracle):
    # repeating phase 0 twice (no alternation) is unstable at r = 4: the pin is sensitive to the offsets
    n, r = 16, 4.0
    T0 = np.stack([oracle.level_1d(e, r, 0) for e in np.eye(n)], axis=1)
    assert _rho(T0 @ T0) > 10.0


# ---- P6/P7: convergence to u = exp(-pi^2 t) sin(pi x) ----
def _maxerr_1d(oracle, n, k, r, t):
    h = 1.0 / (n + 1)
    tau = r * h * h
    levels = 2 * int(round(t / tau / 2))
    x = np.arange(1, n + 1) * h
    u = oracle.run_1d(np.sin(np.pi * x), r, levels, k=k)
    return np.abs(u - np.exp(-np.pi ** 2 * levels * tau) * np.sin(np.pi * x)).max()


def test_p6_convergence_golden(oracle):
    vals = {}
    for ln in golden_lines("p6_p7_convergence.txt"):
        f = ln.split()
        if f[0] == "maxerr" and f[1] == "1":
            n, k, r, t, v = int(f[2]), int(f[3]), float(f[4]), float(f[5]), float(f[6])
            e = _maxerr_1d(oracle, n, k, r, t)
            vals[(n, k, r)] = e
            assert abs(e - v) < 6e-3 * v, (n, k, r, e, v)
    # observed order (reading R-A9): O(h^2) at fixed r, ~ r^2 at fixed h
    assert 3.8 < vals[(63, 1, 1.0)] / vals[(127, 1, 1.0)] < 4.1
    assert 3.8 < vals[(127, 1, 1.0)] / vals[(255, 1, 1.0)] < 4.1
    assert 3.8 < vals[(255, 1, 4.0)] / vals[(511, 1, 4.0)] < 4.1
    assert 3.5 < vals[(63, 1, 4.0)] / vals[(63, 1, 2.0)] < 4.5


def test_p7_config1_end_state(oracle):
    g = dict(ln.split() for ln in golden_lines("p6_p7_convergence.txt") if ln.startswith("c1_"))
    n, r = 64, 1.0
    x = np.arange(1, n + 1) / (n + 1.0)
    u2 = oracle.run_1d(np.sin(np.pi * x), r, 2)
    assert abs(u2[0] - float(g["c1_level2_u1"])) < 1e-15 and abs(u2[63] - float(g["c1_level2_u1"])) < 1e-15
    assert abs(u2[31] - float(g["c1_level2_u32"])) < 1e-14
    u = oracle.run_1d(np.sin(np.pi * x), r, 1000)
    ex = np.exp(-np.pi ** 2 * 1000 / 65.0 ** 2) * np.sin(np.pi * x)
    assert abs(np.abs(u - ex).max() - float(g["c1_maxerr"])) < 1e-8
    assert abs(ex.max() - float(g["c1_maxexact"])) < 1e-7
    assert abs(u[31] - float(g["c1_u32"])) < 1e-11
    assert abs(ex[31] - float(g["c1_exact32"])) < 1e-11


# ---- P8: k >= N+2 reduces to the classical alternating Saul'yev sweeps ----
def test_p8_saulyev_special_case(oracle):
    rng = np.random.default_rng(5)
    n, r, lo, hi = 11, 1.7, 0.3, -0.4
    u = rng.standard_normal(n)
    old = np.concatenate([[lo], u, [hi]])
    a = old.copy()
    for i in range(1, n + 1):                       # scheme A, left to right
        a[i] = (r * a[i - 1] + (1 - r) * old[i] + r * old[i + 1]) / (1 + r)
    np.testing.assert_allclose(oracle.level_1d(u, r, 0, lo, hi, k=n + 2), a[1:-1], rtol=1e-14)
    b = a.copy()
    for i in range(n, 0, -1):                       # scheme B, right to left
        b[i] = (r * b[i + 1] + (1 - r) * a[i] + r * a[i - 1]) / (1 + r)
    np.testing.assert_allclose(oracle.level_1d(a[1:-1], r, 1, lo, hi, k=n + 2), b[1:-1], rtol=1e-14)


# ---- P10: form independence (literal-with-division vs the factored form the kernels use) ----
def test_p10_factored_form_agrees_in_fp64(oracle):
    rng = np.random.default_rng(11)
    n, r, steps, lo, hi = 512, 4.0, 2000, 0.2, -0.1
    u0 = rng.standard_normal(n)
    ref = oracle.run_1d(u0, r, steps, lo, hi)
    g, e = r / (1 + 2 * r), r / (1 + r)
    v = np.concatenate([[lo], u0, [hi]])
    for s in range(steps):
        ph = s % 2
        new = v.copy()
        left = np.arange(1 + ph, n, 2)              # left members i with i+1 <= n
        p = v[left] + r * (v[left - 1] - v[left])
        q = v[left + 1] + r * (v[left + 2] - v[left + 1])
        w = g * (q - p)
        new[left], new[left + 1] = p + w, q - w
        if ph == 1:
            new[1] = v[1] + e * ((lo - v[1]) + (v[2] - v[1]))
            new[n] = v[n] + e * ((hi - v[n]) + (v[n - 1] - v[n]))
        v = new
    assert np.abs(v[1:-1] - ref).max() / np.abs(ref).max() < 1e-13


def test_level0_sets_starting_phase(oracle):
    u = np.random.default_rng(3).standard_normal(10)
    a = oracle.run_1d(u, 2.0, 3, level0=1)
    b = oracle.level_1d(oracle.level_1d(oracle.level_1d(u, 2.0, 1), 2.0, 0), 2.0, 1)
    np.testing.assert_array_equal(a, b)


def test_batched_equals_loop(oracle):
    rng = np.random.default_rng(9)
    u = rng.standard_normal((5, 12))
    r = rng.uniform(0.5, 8, 5)
    lo, hi = rng.uniform(0, 1, 5), rng.uniform(0, 1, 5)
    out = oracle.run_batched_1d(u, r, 7, lo, hi)
    for b in range(5):
        np.testing.assert_array_equal(out[b], oracle.run_1d(u[b], r[b], 7, lo[b], hi[b]))
