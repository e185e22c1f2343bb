"""Thin Python binding of libge (include/ge.h): argument marshalling only.

Every function has the C entry point's name and forwards to it through ctypes;
every level of the GE scheme is computed by the CUDA kernels
in csrc/.  PyTorch is used by callers for device buffers and streams only:
pass `tensor.data_ptr()` and `torch.cuda.current_stream().cuda_stream`.

There is NO CPU fallback: if libge.so is missing or cannot be loaded, `load()`
raises.  This module imports nothing from oracle/.
"""
from __future__ import annotations

import ctypes
import os
from typing import Optional, Sequence

_HERE = os.path.dirname(os.path.abspath(__file__))
# LIBGE_PATH overrides the in-tree location (e.g. to compare two builds); it must still be a libge.so
LIB_PATH = os.environ.get("LIBGE_PATH") or os.path.join(_HERE, "lib", "libge.so")

GE_F32, GE_F64 = 0, 1
GE_KERNEL_AUTO, GE_KERNEL_PER_STEP, GE_KERNEL_TEMPORAL, GE_KERNEL_PERSISTENT = 0, 1, 2, 3
GE_OK, GE_EINVAL, GE_ENOMEM, GE_ECUDA, GE_EUNSUPPORTED = 0, -1, -2, -3, -4
GE_INFO_KERNEL, GE_INFO_TB, GE_INFO_LAUNCHES, GE_INFO_TILE_VALID, GE_INFO_TILE_LOADED = 0, 1, 2, 3, 4
(GE_INFO_RESIDENT_PATH, GE_INFO_RESIDENT_C, GE_INFO_RESIDENT_WARPS, GE_INFO_RESIDENT_CAPACITY,
 GE_INFO_RESIDENT_TB, GE_INFO_MEETINGS, GE_INFO_SYNC_FAULT, GE_INFO_TEMPORAL_C) = 5, 6, 7, 8, 9, 10, 11, 12
GE_TUNE_TEMPORAL_C, GE_TUNE_TB, GE_TUNE_SEG_PAIRS = 0, 1, 2
GE_TUNE_RESIDENT_C, GE_TUNE_HALO_LANES, GE_TUNE_SYNC_MODE, GE_TUNE_STRIP_COOP, GE_TUNE_FORM_3D, GE_TUNE_K_FORM = 3, 4, 5, 6, 7, 8
GE_TUNE_SRC_FORM = 9
GE_SYNC_FLAGS, GE_SYNC_GRID, GE_SYNC_LINES, GE_SYNC_STAGGER = 0, 1, 2, 3
GE_SYNC_CLUSTER2, GE_SYNC_CLUSTER4, GE_SYNC_CLUSTER8, GE_SYNC_CLUSTER16 = 4, 5, 6, 7

KERNEL_NAMES = {0: "auto", 1: "per_step", 2: "temporal", 3: "persistent"}
_KERNEL_IDS = {v: k for k, v in KERNEL_NAMES.items()}
_DTYPES = {"f32": GE_F32, "f64": GE_F64}

# every symbol include/ge.h declares
EXPORTS = ("ge_plan_create", "ge_step_1d", "ge_step_1d_src", "ge_run_src", "ge_step_1d_var", "ge_run_var", "ge_step_2d", "ge_step_3d", "ge_run", "ge_run_host",
           "ge_plan_get_level", "ge_plan_set_level", "ge_plan_info", "ge_plan_tune", "ge_plan_destroy",
           "ge_fma_probe", "ge_fma_probe_ex", "ge_run_1d_static", "ge_static_limit", "ge_static_error", "ge_strerror", "ge_version")


class ge_desc(ctypes.Structure):
    _fields_ = [
        ("dim", ctypes.c_int32),
        ("nx", ctypes.c_int64), ("ny", ctypes.c_int64),
        ("batch", ctypes.c_int64),
        ("dtype", ctypes.c_int32),
        ("group_k", ctypes.c_int32),
        ("r", ctypes.POINTER(ctypes.c_double)),
        ("bc_lo", ctypes.POINTER(ctypes.c_double)),
        ("bc_hi", ctypes.POINTER(ctypes.c_double)),
        ("kernel", ctypes.c_int32),
        ("tb", ctypes.c_int32),
        ("nz", ctypes.c_int64),
    ]


class GeError(RuntimeError):
    def __init__(self, status: int, where: str):
        self.status = status
        super().__init__("%s: %s (status %d)" % (where, strerror(status), status))


_lib = None


def load() -> ctypes.CDLL:
    """dlopen libge.so; raises if the CUDA library has not been built."""
    global _lib
    if _lib is not None:
        return _lib
    if not os.path.exists(LIB_PATH):
        raise RuntimeError(
            "libge.so is missing (%s): build it with `python -m paper_1310_3422_b200.build`; "
            "there is no CPU fallback" % LIB_PATH)
    lib = ctypes.CDLL(LIB_PATH)
    vp, i64, i32 = ctypes.c_void_p, ctypes.c_int64, ctypes.c_int32
    lib.ge_plan_create.argtypes = [ctypes.POINTER(vp), ctypes.POINTER(ge_desc), vp]
    lib.ge_step_1d.argtypes = [vp, vp, vp, vp]
    lib.ge_step_2d.argtypes = [vp, vp, vp, vp]
    lib.ge_step_3d.argtypes = [vp, vp, vp, vp]
    lib.ge_step_1d_src.argtypes = [vp, vp, vp, vp, ctypes.POINTER(ctypes.c_double), vp]
    lib.ge_run.argtypes = [vp, vp, i64, vp]
    lib.ge_step_1d_var.argtypes = [vp, vp, vp, vp, vp]
    lib.ge_run_var.argtypes = [vp, vp, i64, vp, vp]
    lib.ge_run_src.argtypes = [vp, vp, i64, vp, i64, ctypes.POINTER(ctypes.c_double), ctypes.POINTER(ctypes.c_double), vp]
    lib.ge_run_host.argtypes = [vp, vp, i64, vp]
    lib.ge_plan_get_level.argtypes = [vp, ctypes.POINTER(i64)]
    lib.ge_plan_set_level.argtypes = [vp, i64]
    lib.ge_plan_info.argtypes = [vp, i32, ctypes.POINTER(i64)]
    lib.ge_plan_tune.argtypes = [vp, i32, i64]
    lib.ge_plan_destroy.argtypes = [vp]
    lib.ge_fma_probe.argtypes = [i32, i64, vp, ctypes.POINTER(ctypes.c_double), vp]
    lib.ge_fma_probe_ex.argtypes = [i32, i32, i64, vp, ctypes.POINTER(ctypes.c_double), vp]
    lib.ge_run_1d_static.argtypes = [i32, vp, vp, i64, i64, i64, ctypes.c_double, ctypes.c_double, ctypes.c_double, vp]
    lib.ge_static_limit.argtypes = [i32, ctypes.POINTER(i64)]
    lib.ge_static_error.argtypes = [ctypes.c_char_p, i64]
    lib.ge_strerror.argtypes = [ctypes.c_int]
    lib.ge_strerror.restype = ctypes.c_char_p
    lib.ge_version.argtypes = []
    for name in EXPORTS:
        if name not in ("ge_strerror",):
            getattr(lib, name).restype = ctypes.c_int
    _lib = lib
    return lib


def strerror(status: int) -> str:
    return load().ge_strerror(int(status)).decode()


def ge_version() -> int:
    return load().ge_version()


def _darr(values: Sequence[float]):
    vals = [float(v) for v in values]
    return (ctypes.c_double * len(vals))(*vals)


def ge_plan_create(dim: int, nx: int, ny: int = 1, batch: int = 1, dtype="f64", r=(1.0,),
                   bc_lo=(0.0,), bc_hi=(0.0,), group_k: int = 1, kernel="auto", tb: int = 0,
                   stream: int = 0, nz: int = 1) -> int:
    """Returns the opaque plan handle (an integer address)."""
    lib = load()
    ra, lo, hi = _darr(r), _darr(bc_lo), _darr(bc_hi)
    need = batch if dim == 1 else 1
    needb = batch if dim == 1 else dim
    if len(ra) < need or len(lo) < needb or len(hi) < needb:
        raise GeError(GE_EINVAL, "ge_plan_create (host arrays too short)")
    d = ge_desc(dim=dim, nx=nx, ny=ny, batch=batch,
                dtype=_DTYPES[dtype] if isinstance(dtype, str) else int(dtype),
                group_k=group_k, r=ra, bc_lo=lo, bc_hi=hi,
                kernel=_KERNEL_IDS[kernel] if isinstance(kernel, str) else int(kernel), tb=tb, nz=nz)
    out = ctypes.c_void_p()
    rc = lib.ge_plan_create(ctypes.byref(out), ctypes.byref(d), ctypes.c_void_p(stream))
    if rc != GE_OK:
        raise GeError(rc, "ge_plan_create")
    return out.value


def _check(rc: int, where: str):
    if rc != GE_OK:
        raise GeError(rc, where)


def ge_step_1d(plan: int, u_in: int, u_out: int, stream: int = 0):
    _check(load().ge_step_1d(plan, u_in, u_out, stream), "ge_step_1d")


def ge_step_1d_src(plan: int, u_in: int, u_out: int, tau_f: int, bc4: Sequence[float], stream: int = 0):
    """bc4 = (lo_old, lo_new, hi_old, hi_new); tau_f = device pointer or 0."""
    arr = _darr(bc4)
    if len(arr) != 4:
        raise GeError(GE_EINVAL, "ge_step_1d_src (bc4 needs four values)")
    _check(load().ge_step_1d_src(plan, u_in, u_out, tau_f or None, arr, stream), "ge_step_1d_src")


def ge_step_2d(plan: int, u_in: int, u_out: int, stream: int = 0):
    _check(load().ge_step_2d(plan, u_in, u_out, stream), "ge_step_2d")


def ge_step_3d(plan: int, u_in: int, u_out: int, stream: int = 0):
    _check(load().ge_step_3d(plan, u_in, u_out, stream), "ge_step_3d")


def ge_run(plan: int, u: int, steps: int, stream: int = 0):
    _check(load().ge_run(plan, u, steps, stream), "ge_run")


def ge_run_src(plan: int, u: int, steps: int, tau_f: int, f_level_stride: int, bc_lo_t: Sequence[float],
               bc_hi_t: Sequence[float], stream: int = 0):
    """bc_lo_t / bc_hi_t: steps + 1 boundary values (levels 0 .. steps of the run); tau_f = device pointer or 0."""
    lo, hi = _darr(bc_lo_t), _darr(bc_hi_t)
    if len(lo) != len(hi) or len(lo) < steps + 1 or len(lo) % (steps + 1):
        raise GeError(GE_EINVAL, "ge_run_src (boundary arrays need batch * (steps + 1) values)")
    _check(load().ge_run_src(plan, u, steps, tau_f or None, f_level_stride, lo, hi, stream), "ge_run_src")


def ge_step_1d_var(plan: int, u_in: int, u_out: int, rl: int, stream: int = 0):
    """rl: device pointer to nx + 1 link numbers tau * a_{j+1/2} / h^2."""
    _check(load().ge_step_1d_var(plan, u_in, u_out, rl, stream), "ge_step_1d_var")


def ge_run_var(plan: int, u: int, steps: int, rl: int, stream: int = 0):
    _check(load().ge_run_var(plan, u, steps, rl, stream), "ge_run_var")


def ge_run_host(plan: int, u_host: int, steps: int, stream: int = 0):
    _check(load().ge_run_host(plan, u_host, steps, stream), "ge_run_host")


def ge_plan_get_level(plan: int) -> int:
    v = ctypes.c_int64()
    _check(load().ge_plan_get_level(plan, ctypes.byref(v)), "ge_plan_get_level")
    return v.value


def ge_plan_set_level(plan: int, level: int):
    _check(load().ge_plan_set_level(plan, level), "ge_plan_set_level")


def ge_plan_info(plan: int, what: int) -> int:
    v = ctypes.c_int64()
    _check(load().ge_plan_info(plan, what, ctypes.byref(v)), "ge_plan_info")
    return v.value


def ge_plan_tune(plan: int, what: int, value: int):
    _check(load().ge_plan_tune(plan, what, value), "ge_plan_tune")


def ge_fma_probe(dtype, iters: int, sink: int, stream: int = 0, variant: int = 0) -> float:
    """Enqueue one launch of the FMA throughput probe; returns the flops of that launch.  variant 1: three distinct
    registers per FMA (ge_fma_probe_ex)."""
    v = ctypes.c_double()
    _check(load().ge_fma_probe_ex(_DTYPES[dtype] if isinstance(dtype, str) else int(dtype), variant, iters, sink,
                                  ctypes.byref(v), stream), "ge_fma_probe_ex")
    return v.value


GE_STATIC_MAX_BYTES = 4 * 1024 * 1024


def ge_static_error() -> str:
    buf = ctypes.create_string_buffer(320)
    load().ge_static_error(buf, len(buf))
    return buf.value.decode()


def ge_static_limit(dtype) -> int:
    """Largest nx ge_run_1d_static takes for `dtype` (also does the per-device set-up)."""
    v = ctypes.c_int64()
    rc = load().ge_static_limit(_DTYPES[dtype] if isinstance(dtype, str) else int(dtype), ctypes.byref(v))
    if rc != GE_OK:
        raise GeError(rc, "ge_static_limit: " + ge_static_error())
    return v.value


def ge_run_1d_static(dtype, u_in: int, u_out: int, nx: int, steps: int, r: float, bc_lo: float = 0.0,
                     bc_hi: float = 0.0, level0: int = 0, stream: int = 0):
    """`steps` levels of the 1-D two-point-group scheme from u_in to u_out (device pointers) without any
    allocation: the scratch is a fixed array inside libge.so (include/ge.h)."""
    rc = load().ge_run_1d_static(_DTYPES[dtype] if isinstance(dtype, str) else int(dtype), u_in, u_out, nx, steps,
                                 level0, float(r), float(bc_lo), float(bc_hi), stream)
    if rc != GE_OK:
        raise GeError(rc, "ge_run_1d_static: " + ge_static_error())


def ge_plan_destroy(plan: Optional[int]):
    if plan:
        _check(load().ge_plan_destroy(plan), "ge_plan_destroy")


class Plan:
    """Context-manager convenience around a plan handle built from an inputs.py config dict."""

    def __init__(self, cfg: dict, kernel="auto", tb: int = 0, stream: int = 0, group_k: int = 1):
        self.cfg = cfg
        self.handle = ge_plan_create(cfg["dim"], cfg["nx"], cfg["ny"], cfg["batch"], cfg["dtype"],
                                     list(cfg["r"]), list(cfg["bc_lo"]), list(cfg["bc_hi"]),
                                     group_k=group_k, kernel=kernel, tb=tb, stream=stream, nz=cfg.get("nz", 1))

    def __enter__(self):
        return self

    def __exit__(self, *exc):
        self.close()

    def close(self):
        if self.handle:
            ge_plan_destroy(self.handle)
            self.handle = None

    def step(self, u_in: int, u_out: int, stream: int = 0):
        {1: ge_step_1d, 2: ge_step_2d, 3: ge_step_3d}[self.cfg["dim"]](self.handle, u_in, u_out, stream)

    def step_src(self, u_in: int, u_out: int, tau_f: int, bc4, stream: int = 0):
        ge_step_1d_src(self.handle, u_in, u_out, tau_f, bc4, stream)

    def run(self, u: int, steps: int, stream: int = 0):
        ge_run(self.handle, u, steps, stream)

    def run_src(self, u: int, steps: int, tau_f: int, f_level_stride: int, bc_lo_t, bc_hi_t, stream: int = 0):
        ge_run_src(self.handle, u, steps, tau_f, f_level_stride, bc_lo_t, bc_hi_t, stream)

    def step_var(self, u_in: int, u_out: int, rl: int, stream: int = 0):
        ge_step_1d_var(self.handle, u_in, u_out, rl, stream)

    def run_var(self, u: int, steps: int, rl: int, stream: int = 0):
        ge_run_var(self.handle, u, steps, rl, stream)

    def run_host(self, u_host: int, steps: int, stream: int = 0):
        ge_run_host(self.handle, u_host, steps, stream)

    @property
    def level(self) -> int:
        return ge_plan_get_level(self.handle)

    @level.setter
    def level(self, v: int):
        ge_plan_set_level(self.handle, v)

    def tune(self, what: int, value: int):
        ge_plan_tune(self.handle, what, value)

    def info(self) -> dict:
        return dict(kernel=KERNEL_NAMES[ge_plan_info(self.handle, GE_INFO_KERNEL)],
                    tb=ge_plan_info(self.handle, GE_INFO_TB),
                    launches=ge_plan_info(self.handle, GE_INFO_LAUNCHES),
                    tile_valid=ge_plan_info(self.handle, GE_INFO_TILE_VALID),
                    tile_loaded=ge_plan_info(self.handle, GE_INFO_TILE_LOADED),
                    resident_path=ge_plan_info(self.handle, GE_INFO_RESIDENT_PATH),
                    resident_c=ge_plan_info(self.handle, GE_INFO_RESIDENT_C),
                    resident_warps=ge_plan_info(self.handle, GE_INFO_RESIDENT_WARPS),
                    resident_capacity=ge_plan_info(self.handle, GE_INFO_RESIDENT_CAPACITY),
                    resident_tb=ge_plan_info(self.handle, GE_INFO_RESIDENT_TB),
                    meetings=ge_plan_info(self.handle, GE_INFO_MEETINGS),
                    temporal_c=ge_plan_info(self.handle, GE_INFO_TEMPORAL_C))

    def sync_fault(self) -> int:
        """1 if a tile of the whole-chip persistent kernel gave up waiting (synchronises)."""
        return ge_plan_info(self.handle, GE_INFO_SYNC_FAULT)
