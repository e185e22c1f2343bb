"""Long runs against the ORACLE (not kernel against kernel), in the launch configuration bench.py times
(AUTO plan, default tuning).

* C5 is the one BASELINE.json config whose scheme the paper does not define (reading R-2D; PAPER.md:134,
  :228 only claim the extension), so the oracle is its only anchor: the full 1000 levels are compared
  element by element on grids of many strips x many segments (2048^2: 18 x 16 strips/segments in fp32,
  40 x 19 in fp64; a ragged 2040 x 1030), so that every strip / segment seam accumulates its error over the
  whole run; the full 8192^2 x 1000 run is the `slow` test below (GE_RUN_SLOW=1; ~13 min of oracle time per
  dtype, run once per round through gpurun, result kept in profiles/).
* The whole-chip persistent kernel's meeting kinds (flags, flag-in-data lines, staggered lines) have never
  seen a race detector (compute-sanitizer is refused on this pool), so they are marched for C2's full 10 000
  levels -- thousands of meetings -- and compared with the oracle on sampled dependency cones.
"""
import os
import time

import numpy as np
import pytest

from gpu_util import TOL, rel_err, run_gpu, run_oracle, window_1d
from paper_1310_3422_b200 import inputs

pytestmark = pytest.mark.gpu


@pytest.mark.parametrize("dtype", ["f32", "f64"])
@pytest.mark.parametrize("nx,ny", [(2048, 2048), (2040, 1030)])
def test_c5_many_strips_all_levels_against_the_oracle(oracle, dtype, nx, ny):
    cfg = inputs.make_c5(n=nx, ny=ny, steps=1000, dtype=dtype)
    # (the strip kernel explicitly: below 24 MB of state the AUTO plan takes one launch per level)
    got, info = run_gpu(cfg, cfg["steps"], kernel="temporal")
    assert info["kernel"] == "temporal" and info["launches"] < cfg["steps"] // 4, info
    assert nx // info["tile_valid"] >= 15, info           # many strips (the seams are what is being tested)
    ref = run_oracle(oracle, cfg, cfg["steps"])
    err = rel_err(got, ref)
    print("c5 %s %dx%d x 1000 levels: rel_err %.3e (tolerance %.0e), strips of %d valid columns" % (
        dtype, ny, nx, err, TOL[dtype], info["tile_valid"]))
    assert err <= TOL[dtype], err


@pytest.mark.slow
@pytest.mark.skipif(not os.environ.get("GE_RUN_SLOW"), reason="full 8192^2 x 1000 oracle run: set GE_RUN_SLOW=1")
@pytest.mark.parametrize("dtype", ["f32", "f64"])
def test_c5_full_size_all_levels_against_the_oracle(oracle, dtype):
    cfg = inputs.make_c5(dtype=dtype)
    t0 = time.time()
    got, info = run_gpu(cfg, cfg["steps"])
    t1 = time.time()
    ref = run_oracle(oracle, cfg, cfg["steps"])
    t2 = time.time()
    err = rel_err(got, ref)
    msg = "c5 %s 8192x8192 x 1000 levels, AUTO plan (%s, %d launches): rel_err %.3e (tolerance %.0e); gpu %.1f s incl. copies, oracle %.0f s" % (
        dtype, info["kernel"], info["launches"], err, TOL[dtype], t1 - t0, t2 - t1)
    print(msg)
    out = os.path.join(os.path.dirname(os.path.dirname(os.path.abspath(__file__))), "gpurun_out")
    os.makedirs(out, exist_ok=True)
    with open(os.path.join(out, "c5_full_%s.txt" % dtype), "w") as f:
        f.write(msg + "\n")
    assert err <= TOL[dtype], err


_C2_WINDOWS = {}


def _c2_windows(oracle, cfg, w):
    """Oracle values of a few windows after the full run, computed once (6 s each) and shared by the modes."""
    if not _C2_WINDOWS:
        n = cfg["nx"]
        u0 = cfg["u0"].reshape(-1)
        for s in (0, n - w, n // 2 - 32, 333334, 7 * 1792 - 20):        # ends, middle, and two tile seams
            s -= s % 2
            _C2_WINDOWS[s] = window_1d(oracle, u0, cfg["r"][0], cfg["steps"], 0.0, 0.0, s, w)
    return _C2_WINDOWS


@pytest.mark.parametrize("sync", [1, 0, 2, 3, 6])
def test_c2_all_levels_every_meeting_kind_against_the_oracle(oracle, sync):
    """C2 (N = 2^20 fp64, r = 4, 10 000 levels) on the whole-chip persistent kernel: grid barrier (1, the
    default), neighbour flags (0), flag-in-data lines (2), staggered lines (3)."""
    cfg = inputs.make_c2()
    w = 64
    got, info = run_gpu(cfg, cfg["steps"], sync=sync)
    assert info["kernel"] == "persistent" and info["resident_path"] == 2 and info["launches"] == 1, info
    assert info["meetings"] >= 150, info
    got = got.reshape(-1)
    scale = float(np.abs(cfg["u0"]).max())
    worst = 0.0
    for s, ref in _c2_windows(oracle, cfg, w).items():
        worst = max(worst, float(np.abs(got[s:s + w] - ref).max()))
    print("c2 sync %d: %d meetings, worst window error %.3e of max|u0|" % (sync, info["meetings"], worst / scale))
    assert worst / scale <= TOL["f64"], worst
    assert np.isfinite(got).all()


@pytest.mark.parametrize("sync,rtb", [(0, 8), (2, 8), (3, 8), (2, 2), (6, 8), (4, 2)])
def test_whole_chip_many_meetings_against_the_oracle(oracle, sync, rtb):
    """The same kernel with a meeting every 8 (2) levels -- 250 (1000) meetings in 2000 levels -- on a rod of
    ~60 tiles, whole array against the oracle."""
    cfg = inputs.random_rods(1, 100000, "f64", seed=77)
    steps = 2000
    got, info = run_gpu(cfg, steps, kernel="persistent", rtb=rtb, sync=sync, level0=1)
    assert info["resident_path"] == 2 and info["meetings"] >= steps // rtb - 2, info
    ref = run_oracle(oracle, cfg, steps, level0=1)
    assert rel_err(got, ref) <= TOL["f64"]
