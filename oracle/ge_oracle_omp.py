"""ORACLE-SIDE TIMING DRIVER binding (test infrastructure, NOT the product, NOT the parity oracle).

ctypes loader for oracle/ge_ref_omp.c: the all-cores leg of bench.py's cpu_baseline.
The parity oracle is oracle/ge_ref.c (ge_oracle.py); tests/test_oracle_omp.py pins this driver to it bit
for bit.  Only tests/ and bench.py's cpu_baseline leg may import this module.  It imports nothing from
paper_1310_3422_b200.
"""
from __future__ import annotations

import ctypes
import os
import subprocess

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "ge_ref_omp.c")
_LIB = os.path.join(_HERE, "libge_ref_omp.so")
_lib = None

_f64p = np.ctypeslib.ndpointer(dtype=np.float64, flags="C_CONTIGUOUS")
_i64 = ctypes.c_int64
_f64 = ctypes.c_double


def build(force: bool = False) -> str:
    """gcc -O2 -fopenmp, same floating-point flags as the parity oracle (no contraction, no fast-math)."""
    if force or not os.path.exists(_LIB) or os.path.getmtime(_LIB) < os.path.getmtime(_SRC):
        tmp = _LIB + ".tmp.%d" % os.getpid()
        subprocess.check_call(
            ["gcc", "-O2", "-ffp-contract=off", "-fopenmp", "-fPIC", "-shared", "-std=c99",
             "-Wall", "-Wextra", "-o", tmp, _SRC])
        os.replace(tmp, _LIB)
    return _LIB


def _load():
    global _lib
    if _lib is None:
        lib = ctypes.CDLL(build())
        lib.ge_omp_threads.argtypes = []
        lib.ge_omp_threads.restype = ctypes.c_int
        lib.ge_omp_run_1d.argtypes = [_f64p, _i64, _f64, _f64, _f64, _i64, _i64]
        lib.ge_omp_run_1d.restype = ctypes.c_int
        lib.ge_omp_run_batched_1d.argtypes = [_f64p, _i64, _i64, _f64p, _f64p, _f64p, _i64, _i64]
        lib.ge_omp_run_batched_1d.restype = ctypes.c_int
        lib.ge_omp_run_2d.argtypes = [_f64p, _i64, _i64, _f64, _f64p, _i64, _i64]
        lib.ge_omp_run_2d.restype = ctypes.c_int
        _lib = lib
    return _lib


def threads() -> int:
    """Threads the driver will use (OMP_NUM_THREADS or the cores the process may run on)."""
    return int(_load().ge_omp_threads())


def run_1d(u0, r, steps, bc_lo=0.0, bc_hi=0.0, level0=0):
    u = np.array(u0, dtype=np.float64, order="C", copy=True)
    if _load().ge_omp_run_1d(u, u.shape[0], float(r), float(bc_lo), float(bc_hi), int(level0), int(steps)):
        raise MemoryError("ge_omp_run_1d")
    return u


def run_batched_1d(u0, r, steps, bc_lo, bc_hi, level0=0):
    u = np.array(u0, dtype=np.float64, order="C", copy=True)
    b, n = u.shape
    r = np.ascontiguousarray(np.broadcast_to(np.asarray(r, dtype=np.float64), (b,)))
    lo = np.ascontiguousarray(np.broadcast_to(np.asarray(bc_lo, dtype=np.float64), (b,)))
    hi = np.ascontiguousarray(np.broadcast_to(np.asarray(bc_hi, dtype=np.float64), (b,)))
    if _load().ge_omp_run_batched_1d(u, b, n, r, lo, hi, int(level0), int(steps)):
        raise MemoryError("ge_omp_run_batched_1d")
    return u


def run_2d(u0, r, steps, bc=(0.0, 0.0, 0.0, 0.0), level0=0):
    u = np.array(u0, dtype=np.float64, order="C", copy=True)
    ny, nx = u.shape
    bcv = np.asarray(bc, dtype=np.float64).copy()
    if _load().ge_omp_run_2d(u, nx, ny, float(r), bcv, int(level0), int(steps)):
        raise MemoryError("ge_omp_run_2d")
    return u
