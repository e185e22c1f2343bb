"""ge_run_1d_static (include/ge.h): the entry point that allocates nothing -- its scratch (coefficient block +
second copy of the state) is a fixed file-scope device array inside libge.so (csrc/ge_static.cu).

Checked against the existing path (a ge_plan with kernel = per_step, ge_run) on calls in a row that share the
array: different dtypes, lengths, level counts and phases, so that whatever the previous call left in the array
would show.  The file sorts last on purpose (pytest -x: a failure here hides nothing)."""
import numpy as np
import pytest

from gpu_util import TOL, rel_err, run_gpu
from paper_1310_3422_b200 import inputs

pytestmark = pytest.mark.gpu

# (dtype, nx, steps, level0): vector and scalar forms, odd and even level counts, both starting phases
CALLS = [("f64", 5000, 7, 0), ("f32", 1001, 4, 1), ("f64", 5000, 7, 0), ("f32", 4096, 1, 0), ("f64", 37, 12, 1)]


def _static(cfg, steps, level0):
    import torch
    from paper_1310_3422_b200 import libge
    dev = torch.device("cuda:0")
    u_in = torch.from_numpy(np.ascontiguousarray(cfg["u0"]).reshape(-1)).to(dev)
    u_out = torch.full_like(u_in, float("nan"))
    keep = u_in.clone()
    stream = torch.cuda.current_stream(dev).cuda_stream
    libge.ge_run_1d_static(cfg["dtype"], u_in.data_ptr(), u_out.data_ptr(), cfg["nx"], steps, cfg["r"][0],
                           cfg["bc_lo"][0], cfg["bc_hi"][0], level0=level0, stream=stream)
    torch.cuda.synchronize(dev)
    assert torch.equal(u_in, keep)                      # the input is only read
    return u_out.cpu().numpy().reshape(cfg["u0"].shape)


def test_static_entry_point_matches_the_plan_path_on_calls_in_a_row():
    for i, (dtype, nx, steps, level0) in enumerate(CALLS):
        cfg = inputs.random_rods(1, nx, dtype, seed=50 + nx)
        got = _static(cfg, steps, level0)
        ref, info = run_gpu(cfg, steps, kernel="per_step", level0=level0)
        assert info["kernel"] == "per_step"
        assert np.isfinite(got).all()
        assert rel_err(got, ref) <= TOL[dtype], (i, dtype, nx, steps, level0)
        np.testing.assert_array_equal(got, ref)          # the same kernel and coefficients: bit for bit


def test_static_entry_point_limit_zero_levels_and_no_allocation():
    import torch
    from paper_1310_3422_b200 import libge
    dev = torch.device("cuda:0")
    assert libge.ge_static_limit("f64") == libge.GE_STATIC_MAX_BYTES // 8
    assert libge.ge_static_limit("f32") == libge.GE_STATIC_MAX_BYTES // 4
    # the largest rod it takes, against the plan path
    nmax = libge.ge_static_limit("f64")
    cfg = inputs.random_rods(1, nmax, "f64", seed=9)
    got = _static(cfg, 3, 0)
    ref, _ = run_gpu(cfg, 3, kernel="per_step")
    assert rel_err(got, ref) <= TOL["f64"]
    # one node more: a clear error, nothing enqueued, the output untouched
    a = torch.zeros(nmax + 1, dtype=torch.float64, device=dev)
    b = torch.full_like(a, 7.0)
    with pytest.raises(libge.GeError) as ei:
        libge.ge_run_1d_static("f64", a.data_ptr(), b.data_ptr(), nmax + 1, 1, 1.0)
    assert ei.value.status == libge.GE_EINVAL
    assert "exceeds the static scratch array" in str(ei.value) and str(nmax) in str(ei.value)
    torch.cuda.synchronize(dev)
    assert float(b.min()) == 7.0 and float(b.max()) == 7.0
    # overlapping buffers and bad arguments
    for args in ((a.data_ptr(), a.data_ptr(), 16, 1, 1.0), (a.data_ptr(), a.data_ptr() + 64, 16, 1, 1.0),
                 (a.data_ptr(), b.data_ptr(), 0, 1, 1.0), (a.data_ptr(), b.data_ptr(), 16, -1, 1.0),
                 (a.data_ptr(), b.data_ptr(), 16, 1, -2.0), (0, b.data_ptr(), 16, 1, 1.0)):
        with pytest.raises(libge.GeError) as ei:
            libge.ge_run_1d_static("f64", *args)
        assert ei.value.status == libge.GE_EINVAL, args
    # zero levels: a copy
    cfg = inputs.random_rods(1, 300, "f32", seed=3)
    np.testing.assert_array_equal(_static(cfg, 0, 0), cfg["u0"])
    # no device memory is taken by a call (kernels already loaded by the calls above)
    u_in = torch.from_numpy(np.ascontiguousarray(cfg["u0"]).reshape(-1)).to(dev)
    u_out = torch.empty_like(u_in)
    libge.ge_run_1d_static("f32", u_in.data_ptr(), u_out.data_ptr(), 300, 5, 2.0)
    torch.cuda.synchronize(dev)
    free0 = torch.cuda.mem_get_info(dev)[0]
    for _ in range(3):
        libge.ge_run_1d_static("f32", u_in.data_ptr(), u_out.data_ptr(), 300, 5, 2.0)
    torch.cuda.synchronize(dev)
    assert torch.cuda.mem_get_info(dev)[0] >= free0
