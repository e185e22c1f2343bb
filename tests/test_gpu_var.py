"""GPU parity for ge_step_1d_var / ge_run_var (variable diffusivity, reading R-VAR)
against oracle/ge_ref.c ge_ref_level_1d_var, element by element."""
import numpy as np
import pytest

from gpu_util import TOL, run_gpu
from paper_1310_3422_b200 import inputs

pytestmark = pytest.mark.gpu
_NP = {"f32": np.float32, "f64": np.float64}


def _run(cfg, rl, steps, level0, via="run"):
    import torch
    from paper_1310_3422_b200 import libge
    dev = torch.device("cuda:0")
    u = torch.from_numpy(cfg["u0"].reshape(-1).copy()).to(dev)
    d_rl = torch.from_numpy(rl).to(dev)
    s = torch.cuda.current_stream(dev).cuda_stream
    with libge.Plan(cfg, stream=s) as plan:
        plan.level = level0
        if via == "run":
            plan.run_var(u.data_ptr(), steps, d_rl.data_ptr(), s)
        else:
            v = torch.empty_like(u)
            for _ in range(steps):
                plan.step_var(u.data_ptr(), v.data_ptr(), d_rl.data_ptr(), s)
                u, v = v, u
        torch.cuda.synchronize(dev)
        # ge_run_var is temporally blocked (20 levels per launch in registers, ge_temporal_src.cuh; 16 in shared memory,
        # ge_window.cuh, for rows that are not whole vectors or hold no tile), ge_step_1d_var one launch per level
        n, dtype = cfg["nx"], cfg["dtype"]
        regs = n % (2 if dtype == "f64" else 4) == 0 and n >= (256 if dtype == "f64" else 512)
        assert plan.level == level0 + steps and plan.info()["launches"] == (-(-steps // (20 if regs else 16)) if via == "run" else steps)
    return u.cpu().numpy().astype(np.float64)


@pytest.mark.parametrize("dtype", ["f64", "f32"])
@pytest.mark.parametrize("n", [1, 2, 3, 8, 9, 1000, 4099, 65536])
def test_var_matches_the_oracle(oracle, dtype, n):
    """Random link numbers spread over [0.5, 8] (rounded to the working dtype first, so both sides see the same
    data), unequal boundary values, both starting phases, odd and even level counts, step and run entry points."""
    cfg = inputs.random_rods(1, n, dtype, seed=n + 1)
    rng = np.random.default_rng(n + 2)
    rl = rng.uniform(0.5, 8.0, n + 1).astype(_NP[dtype])
    for level0, steps, via in ((0, 1, "step"), (1, 6, "run"), (0, 41, "run")):
        got = _run(cfg, rl, steps, level0, via)
        ref = oracle.run_1d_var(cfg["u0"].reshape(-1).astype(np.float64), rl.astype(np.float64), steps,
                                cfg["bc_lo"][0], cfg["bc_hi"][0], level0=level0)
        scale = max(np.abs(ref).max(), abs(cfg["bc_lo"][0]), abs(cfg["bc_hi"][0]))
        assert np.abs(got - ref).max() / scale <= TOL[dtype], (n, level0, steps)


def test_constant_links_are_the_plain_scheme(oracle):
    """rl[j] = r everywhere: the level of the paper's Eqs (1)-(4), i.e. the per-level kernel -- to rounding (g is
    computed in the kernel here, on the host there)."""
    for dtype in ("f64", "f32"):
        cfg = inputs.random_rods(1, 5000, dtype, seed=3)
        rl = np.full(5001, cfg["r"][0]).astype(_NP[dtype])
        got = _run(cfg, rl, 20, 0)
        same, _ = run_gpu(cfg, 20, kernel="per_step")
        assert np.abs(got - same.reshape(-1)).max() <= (1e-13 if dtype == "f64" else 2e-5)


def test_long_run_with_a_smooth_coefficient(oracle):
    """a(x) = 1 + x on N = 4095, r = 2, 2000 levels in fp32 and fp64: the tolerance holds over a long run."""
    n = 4095
    h = 1.0 / (n + 1)
    x = np.arange(1, n + 1) * h
    for dtype in ("f64", "f32"):
        rl = (2.0 * (1.0 + (np.arange(n + 1) + 0.5) * h)).astype(_NP[dtype])
        cfg = dict(inputs.random_rods(1, n, dtype), bc_lo=np.array([0.0]), bc_hi=np.array([1.0]),
                   u0=(x + 0.1 * np.sin(7 * np.pi * x))[None, :].astype(_NP[dtype]))
        got = _run(cfg, rl, 2000, 0)
        ref = oracle.run_1d_var(cfg["u0"].reshape(-1).astype(np.float64), rl.astype(np.float64), 2000, 0.0, 1.0)
        assert np.abs(got - ref).max() / np.abs(ref).max() <= TOL[dtype]


def test_var_argument_errors():
    import torch
    from paper_1310_3422_b200 import libge
    u = torch.zeros(256, dtype=torch.float64, device="cuda:0")
    with libge.Plan(inputs.random_rods(2, 64, "f64")) as plan:
        with pytest.raises(libge.GeError) as ei:
            plan.step_var(u.data_ptr(), u.data_ptr() + 8 * 128, u.data_ptr())
        assert ei.value.status == libge.GE_EINVAL
    with libge.Plan(inputs.random_rods(1, 64, "f64"), group_k=2) as plan:
        with pytest.raises(libge.GeError) as ei:
            plan.step_var(u.data_ptr(), u.data_ptr() + 8 * 64, u.data_ptr() + 8 * 128)
        assert ei.value.status == libge.GE_EUNSUPPORTED
    with libge.Plan(inputs.random_rods(1, 64, "f64")) as plan:
        with pytest.raises(libge.GeError):
            plan.step_var(u.data_ptr(), u.data_ptr() + 8 * 64, 0)
        with pytest.raises(libge.GeError):
            plan.run_var(u.data_ptr(), -1, u.data_ptr() + 8 * 128)


@pytest.mark.parametrize("form", [1, 0])
@pytest.mark.parametrize("dtype", ["f64", "f32"])
@pytest.mark.parametrize("batch,n,steps,level0", [(1, 100000, 203, 0), (5, 4099, 77, 1), (3, 1980, 40, 0), (2, 7, 33, 1),
                                                  (4, 4096, 50, 1), (3, 1024, 35, 0), (1, 2 ** 16 + 4, 17, 1)])
def test_run_var_blocked_and_batched(oracle, dtype, batch, n, steps, level0, form):
    """ge_run_var, 16 levels per launch -- form 1 (default): the state, the link numbers and the pair factors of a tile
    in registers (rows of whole aligned vectors that hold a tile); form 0 and every other row: windows of the rods
    with their link numbers in shared memory; batched rods each with its own links and boundary values; several tiles
    / windows per rod, odd and tiny N.  Against the oracle, against the per-level kernel (same expressions: bit for
    bit) and form against form."""
    import torch
    from paper_1310_3422_b200 import libge
    dt = _NP[dtype]
    cfg = inputs.random_rods(batch, n, dtype, seed=n + steps)
    rl = np.random.default_rng(n).uniform(0.5, 8.0, (batch, n + 1)).astype(dt)
    dev = torch.device("cuda:0")
    u = torch.from_numpy(cfg["u0"].copy()).to(dev)
    d_rl = torch.from_numpy(rl).to(dev)
    s = torch.cuda.current_stream(dev).cuda_stream
    with libge.Plan(cfg, stream=s) as plan:
        plan.tune(libge.GE_TUNE_SRC_FORM, form)
        plan.level = level0
        plan.run_var(u.data_ptr(), steps, d_rl.data_ptr(), s)
        torch.cuda.synchronize(dev)
        # 20 levels per launch in registers (rows of whole vectors that hold a tile), 16 in shared memory
        regs = form == 1 and n % (2 if dtype == "f64" else 4) == 0 and n >= (256 if dtype == "f64" else 512)
        assert plan.info()["launches"] == -(-steps // (20 if regs else 16))
        if form == 1:
            v2 = torch.from_numpy(cfg["u0"].copy()).to(dev)
            plan.tune(libge.GE_TUNE_SRC_FORM, 0)
            plan.level = level0
            plan.run_var(v2.data_ptr(), steps, d_rl.data_ptr(), s)
            torch.cuda.synchronize(dev)
            assert torch.equal(u, v2)
    got = u.cpu().numpy().astype(np.float64)
    for b in range(batch):
        ref = oracle.run_1d_var(cfg["u0"][b].astype(np.float64), rl[b].astype(np.float64), steps, cfg["bc_lo"][b],
                                cfg["bc_hi"][b], level0=level0)
        scale = max(np.abs(ref).max(), abs(cfg["bc_lo"][b]), abs(cfg["bc_hi"][b]))
        assert np.abs(got[b] - ref).max() / scale <= TOL[dtype], (b, n, steps)
    if batch == 1:
        one = dict(cfg)
        v = torch.from_numpy(cfg["u0"].reshape(-1).copy()).to(dev)
        w = torch.empty_like(v)
        with libge.Plan(one, stream=s) as plan:
            plan.level = level0
            for _ in range(steps):
                plan.step_var(v.data_ptr(), w.data_ptr(), d_rl.data_ptr(), s)
                v, w = w, v
            torch.cuda.synchronize(dev)
        np.testing.assert_array_equal(v.cpu().numpy(), u.cpu().numpy().reshape(-1))
