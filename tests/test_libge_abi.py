"""CPU-only checks of the boundary: libge.so builds for sm_100a, loads, and exports every symbol
include/ge.h declares.  No compute calls (there is no GPU here)."""
import ctypes
import os
import re

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def lib():
    from paper_1310_3422_b200 import build, libge
    build.build()
    return libge.load()


def _declared():
    src = open(os.path.join(ROOT, "include", "ge.h")).read()
    src = re.sub(r"/\*.*?\*/", "", src, flags=re.S)
    return sorted(set(re.findall(r"\b(ge_[a-z0-9_]+)\s*\(", src)))


def test_header_symbols_are_exported(lib):
    from paper_1310_3422_b200 import libge
    names = _declared()
    assert "ge_plan_create" in names and "ge_run" in names and "ge_step_2d" in names
    for n in names:
        assert hasattr(lib, n), n
    assert sorted(libge.EXPORTS) == names


def test_version_and_strerror(lib):
    from paper_1310_3422_b200 import libge
    assert libge.ge_version() >= 100
    assert libge.strerror(0) == "ok"
    assert "invalid" in libge.strerror(libge.GE_EINVAL)
    assert "group_k" in libge.strerror(libge.GE_EUNSUPPORTED)


def test_validation_needs_no_gpu(lib):
    from paper_1310_3422_b200 import libge
    # argument errors are reported before any CUDA call
    for kw in (dict(dim=4, nx=8), dict(dim=3, nx=8, ny=8, nz=0, bc_lo=(0, 0, 0), bc_hi=(0, 0, 0)), dict(dim=2, nx=8, ny=8, nz=4, bc_lo=(0, 0), bc_hi=(0, 0)), dict(dim=1, nx=0), dict(dim=1, nx=8, r=(-1.0,)),
               dict(dim=1, nx=8, r=(float("nan"),)), dict(dim=2, nx=8, ny=8, batch=2, bc_lo=(0, 0), bc_hi=(0, 0)),
               dict(dim=1, nx=8, ny=2), dict(dim=1, nx=8, group_k=0), dict(dim=1, nx=8, tb=-1),
               dict(dim=2, nx=8, ny=8, group_k=2, bc_lo=(0, 0), bc_hi=(0, 0))):
        with pytest.raises(libge.GeError) as ei:
            libge.ge_plan_create(**kw)
        assert ei.value.status == libge.GE_EINVAL, kw
    with pytest.raises(libge.GeError) as ei:
        libge.ge_plan_create(dim=1, nx=62, group_k=100000)
    assert ei.value.status == libge.GE_EUNSUPPORTED
    assert lib.ge_run(None, None, 1, None) == libge.GE_EINVAL
    assert lib.ge_plan_destroy(None) == libge.GE_EINVAL


def test_desc_struct_layout_matches_header():
    from paper_1310_3422_b200 import libge
    # C layout: int32 dim, (pad), int64 nx, ny, batch, int32 dtype, int32 group_k, 3 pointers, int32 kernel, tb
    assert libge.ge_desc.nx.offset == 8 and libge.ge_desc.batch.offset == 24
    assert libge.ge_desc.dtype.offset == 32 and libge.ge_desc.group_k.offset == 36
    assert libge.ge_desc.r.offset == 40 and libge.ge_desc.kernel.offset == 64
    assert libge.ge_desc.nz.offset == 72
    assert ctypes.sizeof(libge.ge_desc) == 80


def test_product_does_not_import_oracle():
    pkg = os.path.join(ROOT, "paper_1310_3422_b200")
    for dp, _, fs in os.walk(pkg):
        for f in fs:
            if f.endswith((".py", ".cu", ".cuh", ".h")):
                txt = open(os.path.join(dp, f)).read()
                assert "ge_oracle" not in txt and "ge_ref" not in txt, f
    o = open(os.path.join(ROOT, "oracle", "ge_oracle.py")).read()
    assert not re.search(r"^\s*(import|from)\s+paper_1310_3422_b200", o, flags=re.M)


def test_static_entry_point_validates_without_a_gpu(lib):
    """ge_run_1d_static rejects what it cannot take before any CUDA call, with a message that names the limit."""
    from paper_1310_3422_b200 import libge
    assert libge.GE_STATIC_MAX_BYTES == 4 * 1024 * 1024
    for dtype, nmax in ((libge.GE_F64, libge.GE_STATIC_MAX_BYTES // 8), (libge.GE_F32, libge.GE_STATIC_MAX_BYTES // 4)):
        rc = lib.ge_run_1d_static(dtype, 4096, 1 << 30, nmax + 1, 1, 0, 1.0, 0.0, 0.0, None)
        assert rc == libge.GE_EINVAL
        msg = libge.ge_static_error()
        assert "exceeds the static scratch array" in msg and str(nmax) in msg, msg
    for args in ((7, 4096, 8192, 16, 1, 0, 1.0, 0.0, 0.0), (libge.GE_F64, 0, 8192, 16, 1, 0, 1.0, 0.0, 0.0),
                 (libge.GE_F64, 4096, 4096 + 64, 16, 1, 0, 1.0, 0.0, 0.0), (libge.GE_F64, 4096, 8192, 16, -1, 0, 1.0, 0.0, 0.0),
                 (libge.GE_F64, 4096, 8192, 16, 1, 0, 0.0, 0.0, 0.0), (libge.GE_F64, 4096, 8192, 16, 1, 0, 1.0, float("nan"), 0.0),
                 (libge.GE_F64, 4100, 8192, 16, 1, 0, 1.0, 0.0, 0.0)):
        assert lib.ge_run_1d_static(*args, None) == libge.GE_EINVAL, args
        assert libge.ge_static_error() != "ok"
    assert lib.ge_static_error(None, 10) == libge.GE_EINVAL
