"""The all-cores timing driver (oracle/ge_ref_omp.c, bench.py's cpu_baseline leg) against the parity
oracle (oracle/ge_ref.c): the same literal formulas with the loop over a level's groups split across
threads, so the results must be bit-identical -- any N (odd, tiny), both starting phases, odd level
counts, unequal boundary values, batched rods with per-rod r, 2-D with four edge values."""
import numpy as np
import pytest

from paper_1310_3422_b200 import inputs


@pytest.fixture(scope="module")
def omp():
    from oracle import ge_oracle_omp
    ge_oracle_omp.build()
    return ge_oracle_omp


def test_threads_reported(omp):
    assert omp.threads() >= 1


@pytest.mark.parametrize("n", [1, 2, 3, 4, 7, 64, 1001, 4096])
def test_1d_equals_scalar_oracle(oracle, omp, n):
    cfg = inputs.random_rods(1, n, "f64", seed=n)
    for level0, steps in ((0, 1), (1, 1), (0, 2), (1, 7), (0, 40)):
        a = oracle.run_1d(cfg["u0"][0], cfg["r"][0], steps, cfg["bc_lo"][0], cfg["bc_hi"][0], level0=level0)
        b = omp.run_1d(cfg["u0"][0], cfg["r"][0], steps, cfg["bc_lo"][0], cfg["bc_hi"][0], level0=level0)
        np.testing.assert_array_equal(a, b)


def test_batched_equals_scalar_oracle(oracle, omp):
    cfg = inputs.random_rods(37, 513, "f64", seed=4)
    for level0, steps in ((0, 5), (1, 12)):
        a = oracle.run_batched_1d(cfg["u0"], cfg["r"], steps, cfg["bc_lo"], cfg["bc_hi"], level0=level0)
        b = omp.run_batched_1d(cfg["u0"], cfg["r"], steps, cfg["bc_lo"], cfg["bc_hi"], level0=level0)
        np.testing.assert_array_equal(a, b)


@pytest.mark.parametrize("nx,ny", [(1, 1), (2, 2), (3, 5), (8, 8), (65, 34), (130, 67)])
def test_2d_equals_scalar_oracle(oracle, omp, nx, ny):
    cfg = inputs.random_grid(nx, ny, "f64", seed=nx + ny, r=1.7)
    bc = (cfg["bc_lo"][0], cfg["bc_hi"][0], cfg["bc_lo"][1], cfg["bc_hi"][1])
    for level0, steps in ((0, 1), (1, 1), (0, 6), (1, 9)):
        a = oracle.run_2d(cfg["u0"], cfg["r"][0], steps, bc, level0=level0)
        b = omp.run_2d(cfg["u0"], cfg["r"][0], steps, bc, level0=level0)
        np.testing.assert_array_equal(a, b)
