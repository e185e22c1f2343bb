"""ORACLE binding (test infrastructure, NOT the product).

ctypes loader for oracle/ge_ref.c, the plain fp64 CPU statement of the
group-explicit scheme of arXiv 1310.3422.  Only tests/,
__graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs
may import this module.  It imports nothing from paper_1310_3422_b200.

The shared object is built on demand with gcc (-O2, no -ffast-math, no
-ffp-contract: the literal formulas are evaluated as written).
"""
from __future__ import annotations

import ctypes
import os
import subprocess

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "ge_ref.c")
_LIB = os.path.join(_HERE, "libge_ref.so")
_lib = None

_f64p = np.ctypeslib.ndpointer(dtype=np.float64, flags="C_CONTIGUOUS")
_i64 = ctypes.c_int64
_f64 = ctypes.c_double


def build(force: bool = False) -> str:
    """Compile oracle/ge_ref.c into oracle/libge_ref.so (gcc, -O2)."""
    if force or not os.path.exists(_LIB) or os.path.getmtime(_LIB) < os.path.getmtime(_SRC):
        tmp = _LIB + ".tmp.%d" % os.getpid()
        subprocess.check_call(
            ["gcc", "-O2", "-ffp-contract=off", "-fPIC", "-shared", "-std=c99",
             "-Wall", "-Wextra", "-o", tmp, _SRC])
        os.replace(tmp, _LIB)
    return _LIB


def _load():
    global _lib
    if _lib is None:
        lib = ctypes.CDLL(build())
        lib.ge_ref_level_1d.argtypes = [_f64p, _f64p, _i64, _f64, _i64, _i64]
        lib.ge_ref_level_1d.restype = None
        lib.ge_ref_level_1d_src.argtypes = [_f64p, _f64p, _i64, _f64, _i64, _i64, ctypes.c_void_p, _f64, _f64]
        lib.ge_ref_level_1d_src.restype = None
        lib.ge_ref_run_1d.argtypes = [_f64p, _i64, _f64, _i64, _f64, _f64, _i64, _i64]
        lib.ge_ref_run_1d.restype = ctypes.c_int
        lib.ge_ref_run_batched_1d.argtypes = [_f64p, _i64, _i64, _f64p, _i64, _f64p, _f64p, _i64, _i64]
        lib.ge_ref_run_batched_1d.restype = ctypes.c_int
        lib.ge_ref_level_1d_var.argtypes = [_f64p, _f64p, _i64, _f64p, _i64, _i64]
        lib.ge_ref_level_1d_var.restype = None
        lib.ge_ref_run_1d_var.argtypes = [_f64p, _i64, _f64p, _i64, _f64, _f64, _i64, _i64]
        lib.ge_ref_run_1d_var.restype = ctypes.c_int
        lib.ge_ref_level_2d.argtypes = [_f64p, _f64p, _i64, _i64, _f64, _i64]
        lib.ge_ref_level_2d.restype = None
        lib.ge_ref_run_2d.argtypes = [_f64p, _i64, _i64, _f64, _f64p, _i64, _i64]
        lib.ge_ref_run_2d.restype = ctypes.c_int
        lib.ge_ref_level_3d.argtypes = [_f64p, _f64p, _i64, _i64, _i64, _f64, _i64]
        lib.ge_ref_level_3d.restype = None
        lib.ge_ref_run_3d.argtypes = [_f64p, _i64, _i64, _i64, _f64, _f64p, _i64, _i64]
        lib.ge_ref_run_3d.restype = ctypes.c_int
        _lib = lib
    return _lib


def level_1d(u, r, phase, bc_lo=0.0, bc_hi=0.0, k=1):
    """One level: interior values u[0..N-1] (nodes 1..N) -> new interior values."""
    u = np.asarray(u, dtype=np.float64)
    n = u.shape[0]
    old = np.empty(n + 2, dtype=np.float64)
    old[0], old[-1] = bc_lo, bc_hi
    old[1:-1] = u
    new = np.empty_like(old)
    _load().ge_ref_level_1d(old, new, n, float(r), int(k), int(phase))
    return new[1:-1].copy()


def level_1d_src(u, r, phase, bc_old, bc_new, s=None, k=1):
    """One level with a source term and moving boundary values (reading R-N3): bc_old = (lo, hi)
    at the old level, bc_new at the new level, s[i] = tau*f at interior node i+1 (or None)."""
    u = np.asarray(u, dtype=np.float64)
    n = u.shape[0]
    old = np.empty(n + 2, dtype=np.float64)
    old[0], old[-1] = bc_old
    old[1:-1] = u
    new = np.empty_like(old)
    sp = None
    if s is not None:
        sp = np.zeros(n + 2, dtype=np.float64)
        sp[1:-1] = np.asarray(s, dtype=np.float64)
    _load().ge_ref_level_1d_src(old, new, n, float(r), int(k), int(phase),
                                sp.ctypes.data if sp is not None else None, float(bc_new[0]), float(bc_new[1]))
    return new[1:-1].copy()


def level_1d_var(u, rl, phase, bc_lo=0.0, bc_hi=0.0, k=1):
    """One level with variable diffusivity (reading R-VAR): rl[j] = tau a_{j+1/2} / h^2 for the link between
    nodes j and j+1, j = 0..N (N+1 numbers)."""
    u = np.asarray(u, dtype=np.float64)
    n = u.shape[0]
    rl = np.ascontiguousarray(rl, dtype=np.float64)
    assert rl.shape == (n + 1,)
    old = np.empty(n + 2, dtype=np.float64)
    old[0], old[-1] = bc_lo, bc_hi
    old[1:-1] = u
    new = np.empty_like(old)
    _load().ge_ref_level_1d_var(old, new, n, rl, int(k), int(phase))
    return new[1:-1].copy()


def run_1d_var(u0, rl, steps, bc_lo=0.0, bc_hi=0.0, k=1, level0=0):
    u = np.array(u0, dtype=np.float64, order="C", copy=True)
    rl = np.ascontiguousarray(rl, dtype=np.float64)
    assert rl.shape == (u.shape[0] + 1,)
    if _load().ge_ref_run_1d_var(u, u.shape[0], rl, int(k), float(bc_lo), float(bc_hi), int(level0), int(steps)):
        raise MemoryError("ge_ref_run_1d_var")
    return u


def run_1d(u0, r, steps, bc_lo=0.0, bc_hi=0.0, k=1, level0=0):
    """`steps` levels of one rod; returns the final interior values (fp64)."""
    u = np.array(u0, dtype=np.float64, order="C", copy=True)
    rc = _load().ge_ref_run_1d(u, u.shape[0], float(r), int(k), float(bc_lo), float(bc_hi),
                               int(level0), int(steps))
    if rc:
        raise MemoryError("ge_ref_run_1d")
    return u


def run_batched_1d(u0, r, steps, bc_lo, bc_hi, k=1, level0=0):
    """u0: [batch][N]; r, bc_lo, bc_hi: [batch].  Returns the final levels (fp64)."""
    u = np.array(u0, dtype=np.float64, order="C", copy=True)
    assert u.ndim == 2
    b, n = u.shape
    r = np.ascontiguousarray(np.broadcast_to(np.asarray(r, dtype=np.float64), (b,)))
    lo = np.ascontiguousarray(np.broadcast_to(np.asarray(bc_lo, dtype=np.float64), (b,)))
    hi = np.ascontiguousarray(np.broadcast_to(np.asarray(bc_hi, dtype=np.float64), (b,)))
    rc = _load().ge_ref_run_batched_1d(u, b, n, r, int(k), lo, hi, int(level0), int(steps))
    if rc:
        raise MemoryError("ge_ref_run_batched_1d")
    return u


def _pad_2d(u, bc):
    ny, nx = u.shape
    a = np.empty((ny + 2, nx + 2), dtype=np.float64)
    a[:, 0], a[:, -1] = bc[0], bc[1]
    a[0, 1:-1], a[-1, 1:-1] = bc[2], bc[3]
    a[1:-1, 1:-1] = u
    return a


def level_2d(u, r, phase, bc=(0.0, 0.0, 0.0, 0.0)):
    """One 2-D level. u: [Ny][Nx] interior, bc = (x_lo, x_hi, y_lo, y_hi)."""
    u = np.asarray(u, dtype=np.float64)
    ny, nx = u.shape
    old = _pad_2d(u, bc)
    new = np.empty_like(old)
    _load().ge_ref_level_2d(old, new, nx, ny, float(r), int(phase))
    return new[1:-1, 1:-1].copy()


def run_2d(u0, r, steps, bc=(0.0, 0.0, 0.0, 0.0), level0=0):
    """`steps` 2-D levels; returns the final interior values (fp64)."""
    u = np.array(u0, dtype=np.float64, order="C", copy=True)
    ny, nx = u.shape
    bcv = np.asarray(bc, dtype=np.float64).copy()
    rc = _load().ge_ref_run_2d(u, nx, ny, float(r), bcv, int(level0), int(steps))
    if rc:
        raise MemoryError("ge_ref_run_2d")
    return u


def run_3d(u0, r, steps, bc=(0.0,) * 6, level0=0):
    """`steps` 3-D levels (reading R-3D); u0: [Nz][Ny][Nx] interior, bc = (x_lo, x_hi, y_lo, y_hi, z_lo, z_hi)."""
    u = np.array(u0, dtype=np.float64, order="C", copy=True)
    nz, ny, nx = u.shape
    bcv = np.asarray(bc, dtype=np.float64).copy()
    rc = _load().ge_ref_run_3d(u, nx, ny, nz, float(r), bcv, int(level0), int(steps))
    if rc:
        raise MemoryError("ge_ref_run_3d")
    return u


def level_3d(u, r, phase, bc=(0.0,) * 6):
    return run_3d(u, r, 1, bc, level0=phase)


def level_3d_padded(old, r, phase):
    """One 3-D level on a padded array [Nz+2][Ny+2][Nx+2] whose faces hold arbitrary boundary data."""
    old = np.ascontiguousarray(old, dtype=np.float64)
    nz, ny, nx = (d - 2 for d in old.shape)
    new = np.empty_like(old)
    _load().ge_ref_level_3d(old, new, nx, ny, nz, float(r), int(phase))
    return new
