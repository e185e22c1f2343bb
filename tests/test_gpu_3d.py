"""GPU parity in 3-D (2x2x2 groups, reading R-3D) against
oracle/ge_ref.c ge_ref_level_3d, element by element, through ge_step_3d / ge_run."""
import numpy as np
import pytest

from gpu_util import TOL, rel_err, run_gpu, run_oracle
from paper_1310_3422_b200 import inputs

pytestmark = pytest.mark.gpu


@pytest.mark.parametrize("dtype", ["f64", "f32"])
@pytest.mark.parametrize("nx,ny,nz", [(1, 1, 1), (2, 2, 2), (3, 3, 3), (4, 4, 4), (5, 4, 3), (2, 7, 4), (8, 8, 8), (65, 33, 10),
                                      (64, 6, 5), (130, 17, 9), (31, 32, 33)])
def test_per_step_3d(oracle, dtype, nx, ny, nz):
    """Full groups (Walsh closed form) and groups cut by faces, edges and corners (both phases, even and
    odd sizes), six different face values."""
    cfg = inputs.random_box(nx, ny, nz, dtype, seed=nx * 100 + ny * 10 + nz, r=1.7)
    for level0 in (0, 1):
        for steps in (1, 2, 7):
            got, info = run_gpu(cfg, steps, level0=level0, form3d=0)
            ref = run_oracle(oracle, cfg, steps, level0=level0)
            assert info["kernel"] == "per_step" and info["launches"] == steps
            assert rel_err(got, ref) <= (5e-14 if dtype == "f64" else 5e-6), (nx, ny, nz, level0, steps)


@pytest.mark.parametrize("dtype", ["f64", "f32"])
@pytest.mark.parametrize("nx,ny,nz", [(8, 8, 8), (10, 9, 8), (64, 12, 9), (66, 40, 24), (65, 33, 11), (130, 17, 70), (200, 31, 32),
                                      (31, 32, 33), (256, 20, 150), (132, 9, 8), (516, 8, 9), (16, 8, 8), (12, 9, 8)])
def test_per_step_3d_streaming(oracle, dtype, nx, ny, nz):
    """The streaming form (default): ge3d_stream_kernel for the deep groups (16-byte pieces when nx is a multiple
    of the nodes a lane holds -- phase 1 then in the shifted form, whose values cross lane and warp edges --, scalar
    form otherwise; several warps in x, z segments, ragged everything; every full group, the face values standing
    in for neighbours outside the box) + ge3d_shell_kernel for the
    outermost layer of groups.  Against the oracle, and bit for bit against the thread-per-group kernel."""
    cfg = inputs.random_box(nx, ny, nz, dtype, seed=nx * 100 + ny * 10 + nz, r=1.7)
    vec = nx % (2 if dtype == "f64" else 4) == 0
    for level0, steps in ((0, 1), (1, 1), (0, 2), (1, 7)):
        # form 2 = the streaming kernel whatever the row length (the default takes it for 16-byte rows only)
        got, info = run_gpu(cfg, steps, level0=level0, form3d=2)
        # one streaming launch per level, one shell launch when the level has groups cut by a face
        cut = sum(1 for lev in range(level0, level0 + steps) if lev % 2 == 1 or nx % 2 or ny % 2 or nz % 2)
        assert info["kernel"] == "per_step" and info["launches"] == steps + cut
        auto, ainfo = run_gpu(cfg, steps, level0=level0)
        assert ainfo["launches"] == (steps + cut if vec else steps), ainfo
        np.testing.assert_array_equal(got, auto)
        ref = run_oracle(oracle, cfg, steps, level0=level0)
        assert rel_err(got, ref) <= (5e-14 if dtype == "f64" else 5e-6), (nx, ny, nz, level0, steps)
        same, _ = run_gpu(cfg, steps, level0=level0, form3d=0)
        np.testing.assert_array_equal(got, same, err_msg=str((nx, ny, nz, level0, steps)))


def test_step_3d_entry_point_and_long_run(oracle):
    cfg = inputs.random_box(24, 20, 18, "f64", seed=8, r=3.0)
    a, _ = run_gpu(cfg, 6, via="step")
    b, _ = run_gpu(cfg, 6, via="run")
    np.testing.assert_array_equal(a, b)
    for dtype in ("f64", "f32"):
        cfg = inputs.make_box(n=32, steps=200, dtype=dtype)
        got, _ = run_gpu(cfg, cfg["steps"])
        assert rel_err(got, run_oracle(oracle, cfg, cfg["steps"])) <= TOL[dtype]


def test_3d_rejects_what_it_does_not_do():
    from paper_1310_3422_b200 import libge
    with pytest.raises(libge.GeError) as ei:
        libge.ge_plan_create(dim=3, nx=8, ny=8, nz=8, group_k=2, bc_lo=(0, 0, 0), bc_hi=(0, 0, 0))
    assert ei.value.status == libge.GE_EINVAL
    with libge.Plan(inputs.random_box(8, 8, 8)) as plan:
        assert plan.info()["kernel"] == "per_step"
        with pytest.raises(libge.GeError):
            libge.ge_step_2d(plan.handle, 1024, 4096)
