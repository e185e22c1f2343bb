"""GPU parity for ge_step_1d_src (source term + time-dependent boundary values; SURVEY.md 8(f) NEXT-3,
DESIGN.md reading R-N3) against oracle/ge_ref.c ge_ref_level_1d_src, element by element."""
import numpy as np
import pytest

from gpu_util import TOL, run_gpu
from paper_1310_3422_b200 import inputs

pytestmark = pytest.mark.gpu
_NP = {"f32": np.float32, "f64": np.float64}


def _march(oracle, cfg, steps, level0, srcs, bcs, use_src=True):
    """GPU and oracle side by side on the same per-level data; returns (gpu, oracle) final levels."""
    import torch
    from paper_1310_3422_b200 import libge
    dt = _NP[cfg["dtype"]]
    dev = torch.device("cuda:0")
    u = torch.from_numpy(cfg["u0"].reshape(-1).copy()).to(dev)
    v = torch.empty_like(u)
    s = torch.cuda.current_stream(dev).cuda_stream
    ref = cfg["u0"].reshape(-1).astype(np.float64)
    r = float(cfg["r"][0])
    with libge.Plan(cfg, kernel="per_step", stream=s) as plan:
        plan.level = level0
        for n in range(steps):
            src = srcs[n].astype(dt)
            lo_o, lo_n, hi_o, hi_n = [float(dt(x)) for x in bcs[n]]       # what the GPU will see
            d_src = torch.from_numpy(src).to(dev)
            plan.step_src(u.data_ptr(), v.data_ptr(), d_src.data_ptr() if use_src else 0, (lo_o, lo_n, hi_o, hi_n), s)
            torch.cuda.synchronize(dev)
            u, v = v, u
            ref = oracle.level_1d_src(ref, r, (level0 + n) % 2, (lo_o, hi_o), (lo_n, hi_n),
                                      src.astype(np.float64) if use_src else None)
        assert plan.level == level0 + steps and plan.info()["launches"] == steps
    return u.cpu().numpy().astype(np.float64), ref


@pytest.mark.parametrize("dtype", ["f64", "f32"])
@pytest.mark.parametrize("n", [1, 2, 3, 8, 9, 1000, 4099, 65536])
def test_step_src_matches_the_oracle(oracle, dtype, n):
    cfg = inputs.random_rods(1, n, dtype, seed=n)
    rng = np.random.default_rng(n + 5)
    for level0 in (0, 1):
        steps = 6
        srcs = [rng.uniform(-0.1, 0.1, n) for _ in range(steps)]
        walk = rng.uniform(-1, 1, (steps + 1, 2))                       # boundary values level by level
        bcs = [(walk[i, 0], walk[i + 1, 0], walk[i, 1], walk[i + 1, 1]) for i in range(steps)]
        got, ref = _march(oracle, cfg, steps, level0, srcs, bcs)
        scale = max(np.abs(ref).max(), np.abs(walk).max())
        assert np.abs(got - ref).max() / scale <= TOL[dtype], (n, level0)


def test_step_src_without_source_and_with_fixed_boundaries_is_the_plain_level(oracle):
    for dtype in ("f64", "f32"):
        cfg = inputs.random_rods(1, 5000, dtype, seed=3)
        lo, hi = float(cfg["bc_lo"][0]), float(cfg["bc_hi"][0])
        for level0 in (0, 1):
            got, _ = _march(oracle, cfg, 5, level0, [np.zeros(5000)] * 5, [(lo, lo, hi, hi)] * 5, use_src=False)
            same, _ = run_gpu(cfg, 5, kernel="per_step", level0=level0)
            np.testing.assert_array_equal(got, same.reshape(-1).astype(np.float64))


def test_manufactured_solution_on_the_gpu(oracle):
    """u = e^{-pi^2 t} sin(pi x) + x t^2 + (1-x) sin t on N = 127, r = 1, to t ~ 0.1: the GPU follows the
    oracle to 1e-12 and the exact solution to the scheme's O(h^2) error."""
    n, r = 127, 1.0
    h = 1.0 / (n + 1)
    x = np.arange(1, n + 1) * h
    tau = r * h * h
    steps = int(round(0.1 / tau)); steps += steps % 2
    exact = lambda t: np.exp(-np.pi ** 2 * t) * np.sin(np.pi * x) + x * t * t + (1 - x) * np.sin(t)
    f = lambda t: 2 * x * t + (1 - x) * np.cos(t)
    cfg = dict(inputs.random_rods(1, n, "f64"), r=np.array([r]), u0=exact(0.0)[None, :].copy())
    ts = [i * tau for i in range(steps + 1)]
    srcs = [tau * f(t + tau / 2) for t in ts[:-1]]
    bcs = [(np.sin(t), np.sin(t + tau), t * t, (t + tau) ** 2) for t in ts[:-1]]
    got, ref = _march(oracle, cfg, steps, 0, srcs, bcs)
    assert np.abs(got - ref).max() <= 1e-12
    err = np.abs(got - exact(ts[-1])).max()
    assert err < 3e-4, err


def test_step_src_argument_errors():
    import torch
    from paper_1310_3422_b200 import libge
    u = torch.zeros(256, dtype=torch.float64, device="cuda:0")
    with libge.Plan(inputs.random_rods(2, 64, "f64")) as plan:            # batched rods: not supported
        with pytest.raises(libge.GeError) as ei:
            plan.step_src(u.data_ptr(), u.data_ptr() + 8 * 128, 0, (0, 0, 0, 0))
        assert ei.value.status == libge.GE_EINVAL
    with libge.Plan(inputs.random_rods(1, 64, "f64"), group_k=2) as plan:
        with pytest.raises(libge.GeError) as ei:
            plan.step_src(u.data_ptr(), u.data_ptr() + 8 * 64, 0, (0, 0, 0, 0))
        assert ei.value.status == libge.GE_EUNSUPPORTED
    with libge.Plan(inputs.random_rods(1, 64, "f64")) as plan:
        with pytest.raises(libge.GeError):
            plan.step_src(u.data_ptr(), u.data_ptr() + 8 * 64, 0, (0, float("nan"), 0, 0))
        with pytest.raises(libge.GeError):
            plan.step_src(u.data_ptr(), u.data_ptr(), 0, (0, 0, 0, 0))


@pytest.mark.parametrize("dtype", ["f64", "f32"])
@pytest.mark.parametrize("n,steps,level0,per_level", [(1000, 7, 0, True), (4099, 12, 1, True), (65536, 9, 0, False), (3, 5, 1, False)])
def test_run_src_matches_the_oracle_marched_level_by_level(oracle, dtype, n, steps, level0, per_level):
    """ge_run_src: the whole run behind one call -- a source array per level (or one stationary source) on the
    device, boundary values as host arrays of steps + 1 entries, odd and even level counts (the result lands in u
    either way), both starting phases."""
    import torch
    from paper_1310_3422_b200 import libge
    dt = _NP[dtype]
    cfg = inputs.random_rods(1, n, dtype, seed=n + steps)
    rng = np.random.default_rng(n)
    srcs = rng.uniform(-0.1, 0.1, (steps if per_level else 1, n)).astype(dt)
    walk = rng.uniform(-1, 1, (steps + 1, 2)).astype(dt).astype(np.float64)
    dev = torch.device("cuda:0")
    u = torch.from_numpy(cfg["u0"].reshape(-1).copy()).to(dev)
    d_src = torch.from_numpy(srcs).to(dev)
    s = torch.cuda.current_stream(dev).cuda_stream
    with libge.Plan(cfg, stream=s) as plan:
        plan.level = level0
        plan.run_src(u.data_ptr(), steps, d_src.data_ptr(), n if per_level else 0, walk[:, 0], walk[:, 1], s)
        torch.cuda.synchronize(dev)
        assert plan.level == level0 + steps
        # a source per level: one launch per level; a stationary source: 16 levels per launch (ge_window.cuh)
        assert plan.info()["launches"] == (steps if per_level else -(-steps // 16))
    ref = cfg["u0"].reshape(-1).astype(np.float64)
    for i in range(steps):
        ref = oracle.level_1d_src(ref, float(cfg["r"][0]), (level0 + i) % 2, (walk[i, 0], walk[i, 1]),
                                  (walk[i + 1, 0], walk[i + 1, 1]), srcs[i if per_level else 0].astype(np.float64))
    scale = max(np.abs(ref).max(), np.abs(walk).max())
    assert np.abs(u.cpu().numpy().astype(np.float64) - ref).max() / scale <= TOL[dtype]


def test_run_src_argument_errors():
    import torch
    from paper_1310_3422_b200 import libge
    u = torch.zeros(256, dtype=torch.float64, device="cuda:0")
    with libge.Plan(inputs.random_rods(1, 64, "f64")) as plan:
        with pytest.raises(libge.GeError):
            plan.run_src(u.data_ptr(), 2, 0, 0, (0, 0), (0, 0, 0))               # boundary arrays too short
        with pytest.raises(libge.GeError):
            plan.run_src(u.data_ptr(), 2, u.data_ptr() + 8 * 64, 10, (0, 0, 0), (0, 0, 0))   # 0 < stride < nx
        with pytest.raises(libge.GeError):
            plan.run_src(u.data_ptr(), 1, 0, 0, (0, float("inf")), (0, 0))
        plan.run_src(u.data_ptr(), 0, 0, 0, (0.0,), (0.0,))
        assert plan.level == 0


@pytest.mark.parametrize("form", [1, 0])
@pytest.mark.parametrize("dtype", ["f64", "f32"])
@pytest.mark.parametrize("batch,n,steps,level0", [(1, 100000, 203, 0), (5, 4099, 77, 1), (3, 1980, 40, 0), (2, 7, 33, 1),
                                                  (64, 4096, 50, 0), (3, 1024, 35, 1), (2, 2 ** 16, 64, 1), (1, 2 ** 16 + 4, 17, 0)])
def test_run_src_blocked_with_a_stationary_source(oracle, dtype, batch, n, steps, level0, form):
    """ge_run_src with one stationary source array: temporally blocked, 16 levels per launch -- form 1 (default): the
    state and the source values of a tile in registers (rows of whole aligned vectors that hold a tile), form 0 and
    every other row: windows of the rods with their source values in shared memory; batched rods with per-rod r,
    boundary values that move every level and differ from rod to rod; several tiles / windows per rod, ragged last
    one, odd and tiny N, both starting phases, odd level counts.  Against the oracle marched level by level, and the
    two forms bit for bit against each other."""
    import torch
    from paper_1310_3422_b200 import libge
    dt = _NP[dtype]
    cfg = inputs.random_rods(batch, n, dtype, seed=n + steps)
    rng = np.random.default_rng(n + batch)
    src = rng.uniform(-0.1, 0.1, (batch, n)).astype(dt)
    walk = (rng.uniform(-1, 1, (batch, 1, 2)) + 0.05 * np.cumsum(rng.uniform(-1, 1, (batch, steps + 1, 2)), axis=1)).astype(dt).astype(np.float64)
    dev = torch.device("cuda:0")
    u = torch.from_numpy(cfg["u0"].copy()).to(dev)
    d_src = torch.from_numpy(src).to(dev)
    s = torch.cuda.current_stream(dev).cuda_stream
    with libge.Plan(cfg, stream=s) as plan:
        plan.tune(libge.GE_TUNE_SRC_FORM, form)
        plan.level = level0
        plan.run_src(u.data_ptr(), steps, d_src.data_ptr(), 0, walk[:, :, 0].reshape(-1), walk[:, :, 1].reshape(-1), s)
        torch.cuda.synchronize(dev)
        # 20 levels per launch in registers (rows of whole vectors that hold a tile), 16 in shared memory
        regs = form == 1 and n % (2 if dtype == "f64" else 4) == 0 and n >= (256 if dtype == "f64" else 512)
        assert plan.level == level0 + steps and plan.info()["launches"] == -(-steps // (20 if regs else 16))
        if form == 1:                       # the other form from the same start: the same bits
            v = torch.from_numpy(cfg["u0"].copy()).to(dev)
            plan.tune(libge.GE_TUNE_SRC_FORM, 0)
            plan.level = level0
            plan.run_src(v.data_ptr(), steps, d_src.data_ptr(), 0, walk[:, :, 0].reshape(-1), walk[:, :, 1].reshape(-1), s)
            torch.cuda.synchronize(dev)
            assert torch.equal(u, v)
    got = u.cpu().numpy().astype(np.float64)
    for b in range(batch):
        ref = cfg["u0"][b].astype(np.float64)
        for i in range(steps):
            ref = oracle.level_1d_src(ref, float(cfg["r"][b]), (level0 + i) % 2, (walk[b, i, 0], walk[b, i, 1]),
                                      (walk[b, i + 1, 0], walk[b, i + 1, 1]), src[b].astype(np.float64))
        scale = max(np.abs(ref).max(), np.abs(walk[b]).max())
        assert np.abs(got[b] - ref).max() / scale <= TOL[dtype], (b, n, steps)
