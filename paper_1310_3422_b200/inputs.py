"""Seeded synthetic inputs for the five BASELINE.json configs (C1..C5).

This module serves BOTH the oracle-side tests and the CUDA path; it holds none
of the method's arithmetic -- only the initial/boundary data recipes of
DESIGN.md "Input recipe".  All draws come from
numpy.random.default_rng(seed) (PCG64) on the host, in the documented order;
the same arrays go to the oracle and to the GPU.

Neither the paper nor BASELINE.json names a dataset: the paper's workload is
one rod with unspecified phi and constant beta;
these synthetic grids stand in for it.

Each maker returns a dict:
  dim, nx, ny, batch, dtype ("f32"/"f64"), steps, r (ndarray[batch] fp64),
  bc_lo, bc_hi (ndarray fp64; 2-D: (x_lo, y_lo) / (x_hi, y_hi)), u0 (ndarray of
  the working dtype, interior nodes only, row-major), name.
Sizes are parameters so that tests can use reduced grids with the same recipe.
"""
from __future__ import annotations

import numpy as np

_DT = {"f32": np.float32, "f64": np.float64}


def _x(n):
    # interior nodes x_i = i*h, h = 1/(n+1)   (reading R-A10)
    return np.arange(1, n + 1, dtype=np.float64) / float(n + 1)


def _cfg(name, dim, nx, ny, batch, dtype, steps, r, lo, hi, u0):
    return dict(name=name, dim=dim, nx=int(nx), ny=int(ny), batch=int(batch), dtype=dtype,
                steps=int(steps), r=np.asarray(r, dtype=np.float64),
                bc_lo=np.asarray(lo, dtype=np.float64), bc_hi=np.asarray(hi, dtype=np.float64),
                u0=np.ascontiguousarray(u0, dtype=_DT[dtype]))


def make_c1(n=64, steps=1000, r=1.0):
    """C1: 1-D, N=64, r=1, 1000 levels, u0 = sin(pi x), zero BC, fp64."""
    return _cfg("c1", 1, n, 1, 1, "f64", steps, [r], [0.0], [0.0], np.sin(np.pi * _x(n)))


def make_c2(n=2 ** 20, steps=10000, r=4.0, seed=0):
    """C2: 1-D, N=2^20, r=4, 10000 levels, u0 = sum_{m=1..16} a_m sin(m pi x),
    a_m = N(0,1)/m drawn in order m = 1..16 from seed 0, zero BC, fp64."""
    rng = np.random.default_rng(seed)
    x = _x(n)
    u0 = np.zeros(n, dtype=np.float64)
    for m in range(1, 17):
        a_m = rng.normal(0.0, 1.0) / m
        u0 += a_m * np.sin(m * np.pi * x)
    return _cfg("c2", 1, n, 1, 1, "f64", steps, [r], [0.0], [0.0], u0)


def make_c3(batch=4096, n=4096, steps=2000, seed=1):
    """C3: batched rods, fp32.  Draw order from seed 1: r (batch) ~ U[0.5, 8],
    u0 (batch x n, row-major) ~ U[0,1], bc_lo (batch) ~ U[0,1], bc_hi (batch) ~ U[0,1].
    r and the boundary values are rounded to fp32-representable numbers so that
    oracle and GPU see identical data (reading R-A8)."""
    rng = np.random.default_rng(seed)
    r = rng.uniform(0.5, 8.0, size=batch).astype(np.float32).astype(np.float64)
    u0 = rng.uniform(0.0, 1.0, size=(batch, n)).astype(np.float32)
    lo = rng.uniform(0.0, 1.0, size=batch).astype(np.float32).astype(np.float64)
    hi = rng.uniform(0.0, 1.0, size=batch).astype(np.float32).astype(np.float64)
    return _cfg("c3", 1, n, 1, batch, "f32", steps, r, lo, hi, u0)


def make_c4(n=2 ** 28, steps=200, r=2.0, seed=2):
    """C4: 1-D, N=2^28, r=2, 200 levels, u0 = sin(pi x) + 0.01 N(0,1) (seed 2), zero BC, fp64."""
    rng = np.random.default_rng(seed)
    u0 = np.sin(np.pi * _x(n))
    u0 += 0.01 * rng.standard_normal(n)
    return _cfg("c4", 1, n, 1, 1, "f64", steps, [r], [0.0], [0.0], u0)


def make_c5(n=8192, steps=1000, r=2.0, dtype="f32", seed=3, ny=None):
    """C5: 2-D, n x n interior, r=2, 1000 levels, u0 = sin(pi x) sin(pi y) + 0.01 N(0,1)
    (seed 3, drawn row-major [j][i]), zero BC on all edges, fp32 or fp64."""
    ny = n if ny is None else ny
    rng = np.random.default_rng(seed)
    u0 = np.outer(np.sin(np.pi * _x(ny)), np.sin(np.pi * _x(n)))
    u0 += 0.01 * rng.standard_normal((ny, n))
    u0 = u0.astype(_DT[dtype])
    return _cfg("c5_" + dtype, 2, n, ny, 1, dtype, steps, [r], [0.0, 0.0], [0.0, 0.0], u0)


def random_rods(batch, n, dtype="f64", seed=1234, r_lo=0.5, r_hi=8.0):
    """Generic seeded case for parity tests: per-rod r, unequal non-zero boundary values."""
    rng = np.random.default_rng(seed)
    t = _DT[dtype]
    r = rng.uniform(r_lo, r_hi, size=batch).astype(t).astype(np.float64)
    u0 = rng.uniform(-1.0, 1.0, size=(batch, n)).astype(t)
    lo = rng.uniform(-1.0, 1.0, size=batch).astype(t).astype(np.float64)
    hi = rng.uniform(-1.0, 1.0, size=batch).astype(t).astype(np.float64)
    return _cfg("rods", 1, n, 1, batch, dtype, 0, r, lo, hi, u0)


def random_grid(nx, ny, dtype="f64", seed=4321, r=2.0):
    """Generic seeded 2-D case for parity tests with four different edge values."""
    rng = np.random.default_rng(seed)
    t = _DT[dtype]
    u0 = rng.uniform(-1.0, 1.0, size=(ny, nx)).astype(t)
    b = rng.uniform(-1.0, 1.0, size=4).astype(t).astype(np.float64)
    return _cfg("grid", 2, nx, ny, 1, dtype, 0, [r], [b[0], b[2]], [b[1], b[3]], u0)


def random_box(nx, ny, nz, dtype="f64", seed=999, r=2.0):
    """Generic seeded 3-D case with six different face values; u0 is [nz][ny][nx]."""
    rng = np.random.default_rng(seed)
    t = _DT[dtype]
    u0 = rng.uniform(-1.0, 1.0, size=(nz, ny, nx)).astype(t)
    b = rng.uniform(-1.0, 1.0, size=6).astype(t).astype(np.float64)
    cfg = _cfg("box", 3, nx, ny, 1, dtype, 0, [r], [b[0], b[2], b[4]], [b[1], b[3], b[5]], u0)
    cfg["nz"] = int(nz)
    return cfg


def make_box(n=512, steps=100, r=2.0, dtype="f32", seed=4):
    """3-D measurement workload (not a BASELINE.json config): n^3 interior, u0 = sin(pi x) sin(pi y)
    sin(pi z) + 0.01 N(0,1) from `seed`, zero boundary values."""
    rng = np.random.default_rng(seed)
    x = np.sin(np.pi * _x(n))
    u0 = x[None, None, :] * x[None, :, None] * x[:, None, None]
    u0 = u0 + 0.01 * rng.standard_normal((n, n, n))
    cfg = _cfg("box", 3, n, n, 1, dtype, steps, [r], [0.0, 0.0, 0.0], [0.0, 0.0, 0.0], u0)
    cfg["nz"] = int(n)
    return cfg


def make_paper(n=8206, steps=1200, r=1.0, dtype="f32"):
    """The paper's own run shape: 8208 nodes including the two boundary nodes, sub-domain
    couples of 32 nodes (k = 16, passed to the plan as group_k), up to ~1200 levels; the paper states
    neither r nor phi: r = 1, u0 = sin(pi x), zero boundary values are this repository's choice."""
    return _cfg("paper", 1, n, 1, 1, dtype, steps, [r], [0.0], [0.0], np.sin(np.pi * _x(n)))
