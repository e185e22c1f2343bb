"""GPU parity at BASELINE.json's FULL sizes, in the launch configuration bench.py times (AUTO plan,
default tuning).  The oracle cannot march 2^28 nodes, so it computes SAMPLED outputs one by one on
their dependency cone (a two-point group reads u_{i-1}..u_{i+2}: the cone widens
by at most 2 nodes per side and level; gpu_util.window_1d / window_2d), or whole sampled rods.
Where the cone of the full run is too large for the oracle (C5: 1000 levels -> 4000^2 nodes per
sample) the sampled check runs the full grid for fewer levels in the same launch configuration, and
the full run is checked through a property that holds at any size: the blocked kernel must agree
bit for bit with the per-level kernel, whose every launch is one oracle-checked level."""
import numpy as np
import pytest

from gpu_util import TOL, rel_err, run_gpu, window_1d, window_2d
from paper_1310_3422_b200 import inputs

pytestmark = pytest.mark.gpu


def _scale(cfg):
    return float(np.abs(cfg["u0"]).max())


def test_c4_full_size_sampled(oracle):
    """C4: N = 2^28 fp64, r = 2, 200 levels -- the default bench workload (TMA-staged temporal kernel)."""
    cfg = inputs.make_c4()
    got, info = run_gpu(cfg, cfg["steps"])
    assert info["kernel"] == "temporal" and info["launches"] < cfg["steps"]
    got = got.reshape(-1)
    n, w = cfg["nx"], 96
    valid = info["tile_valid"]
    rng = np.random.default_rng(11)
    starts = [0, n - w, valid - 40, 7 * valid - 50, (n // valid) * valid - 60, n // 2 - 13]
    starts += [int(s) for s in rng.integers(0, n - w, size=10)]
    u0 = cfg["u0"].reshape(-1)
    worst = 0.0
    for s in starts:
        s -= s % 2
        ref = window_1d(oracle, u0, cfg["r"][0], cfg["steps"], 0.0, 0.0, s, w)
        worst = max(worst, float(np.abs(got[s:s + w] - ref).max()))
    assert worst / _scale(cfg) <= TOL["f64"], worst
    assert np.isfinite(got).all()


def test_c2_full_size_sampled(oracle):
    """C2: N = 2^20 fp64, r = 4, 10 000 levels (whole-chip persistent kernel)."""
    cfg = inputs.make_c2()
    got, info = run_gpu(cfg, cfg["steps"])
    assert info["kernel"] == "persistent" and info["resident_path"] == 2 and info["launches"] == 1
    got = got.reshape(-1)
    n, w = cfg["nx"], 64
    u0 = cfg["u0"].reshape(-1)
    worst = 0.0
    for s in (0, n - w, 524288 - 32, 333334):
        ref = window_1d(oracle, u0, cfg["r"][0], cfg["steps"], 0.0, 0.0, s, w)
        worst = max(worst, float(np.abs(got[s:s + w] - ref).max()))
    assert worst / _scale(cfg) <= TOL["f64"], worst


def test_c3_full_size_sampled_rods(oracle):
    """C3: 4096 rods x 4096 fp32, per-rod r and boundary values, 2000 levels (rod-per-CTA persistent
    kernel): 48 whole rods against the oracle."""
    cfg = inputs.make_c3()
    got, info = run_gpu(cfg, cfg["steps"])
    assert info["kernel"] == "persistent" and info["resident_path"] == 1 and info["launches"] == 1
    rows = np.unique(np.concatenate([[0, 1, 4095], np.random.default_rng(5).integers(0, 4096, size=45)]))
    ref = oracle.run_batched_1d(cfg["u0"][rows].astype(np.float64), cfg["r"][rows], cfg["steps"],
                                cfg["bc_lo"][rows], cfg["bc_hi"][rows])
    err = np.abs(got[rows].astype(np.float64) - ref).max(axis=1) / np.abs(ref).max(axis=1)
    assert err.max() <= TOL["f32"], err.max()
    assert np.isfinite(got).all()


@pytest.mark.parametrize("dtype", ["f32", "f64"])
def test_c5_full_size(oracle, dtype):
    """C5: 8192 x 8192, r = 2.  (a) 96 levels on the full grid in the bench's launch configuration,
    sampled windows against the oracle on their cones; (b) the full 1000 levels: blocked kernel ==
    per-level kernel bit for bit."""
    cfg = inputs.make_c5(dtype=dtype)
    n, w, steps = cfg["nx"], 24, 96
    got, info = run_gpu(cfg, steps)
    assert info["kernel"] == "temporal" and info["launches"] < steps
    valid = info["tile_valid"]
    bc = (0.0, 0.0, 0.0, 0.0)
    rng = np.random.default_rng(3)
    pts = [(0, 0), (n - w, n - w), (0, n - w), (valid - 10, 200), (5 * valid - 14, n - w), (4000, 126), (n - w, 2 * valid - 12)]
    pts += [tuple(int(v) for v in rng.integers(0, n - w, size=2)) for _ in range(5)]
    worst = 0.0
    for x0, y0 in pts:
        x0 -= x0 % 2; y0 -= y0 % 2
        ref = window_2d(oracle, cfg["u0"], cfg["r"][0], steps, bc, x0, y0, w)
        worst = max(worst, float(np.abs(got[y0:y0 + w, x0:x0 + w].astype(np.float64) - ref).max()))
    assert worst / _scale(cfg) <= TOL[dtype], worst
    del got
    a, ia = run_gpu(cfg, cfg["steps"])
    b, ib = run_gpu(cfg, cfg["steps"], kernel="per_step")
    assert ia["launches"] < ib["launches"] == cfg["steps"]
    assert np.isfinite(a).all()
    np.testing.assert_array_equal(a, b)


@pytest.mark.parametrize("dtype,steps,level0", [("f64", 40, 0), ("f32", 33, 1)])
def test_run_host_pipeline_is_bit_identical(dtype, steps, level0):
    """ge_run_host on a rod of several chunks (halo-redundant chunks through a three-slot pipeline) against
    ge_run on the whole rod: bit for bit, including a ragged last chunk and an odd level count."""
    cfg = inputs.random_rods(1, 3 * 2 ** 24 + 40960, dtype, seed=13)
    a, ia = run_gpu(cfg, steps, via="host", level0=level0)
    b, _ = run_gpu(cfg, steps, via="run", level0=level0)
    assert ia["launches"] > 0
    np.testing.assert_array_equal(a, b)


@pytest.mark.parametrize("dtype,kernel", [("f32", "auto"), ("f64", "temporal"), ("f32", "per_step")])
def test_run_host_rod_groups_are_bit_identical(dtype, kernel):
    """ge_run_host on batched rods (eight groups of rods through the three-slot pipeline, ragged last group)
    against ge_run on the whole batch."""
    cfg = inputs.random_rods(1003, 4096, dtype, seed=21)
    a, ia = run_gpu(cfg, 33, via="host", level0=1, kernel=kernel)
    b, ib = run_gpu(cfg, 33, via="run", level0=1, kernel=kernel)
    assert ia["kernel"] == ib["kernel"] and ia["launches"] >= ib["launches"]
    np.testing.assert_array_equal(a, b)
