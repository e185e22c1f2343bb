"""GPU parity: libge (through its C ABI) against the fp64 oracle, element by element, on the
same seeded inputs.  Bar (BASELINE.json north_star): max-abs error relative to max|oracle|
<= 1e-12 (fp64), <= 1e-5 (fp32), measured on the final level (reading R-A7)."""
import numpy as np
import pytest

from gpu_util import TOL, rel_err, rel_err_rows, run_gpu, run_oracle, window_1d, window_2d
from paper_1310_3422_b200 import inputs

pytestmark = pytest.mark.gpu


# ------------------------------------------------------------------ strategy A, 1-D ------
@pytest.mark.parametrize("dtype", ["f64", "f32"])
@pytest.mark.parametrize("n", [1, 2, 3, 4, 7, 8, 64, 1000, 1026, 4099])
def test_per_step_1d_small(oracle, dtype, n):
    cfg = inputs.random_rods(3, n, dtype, seed=100 + n)
    for level0 in (0, 1):
        for steps in (1, 2, 5):
            got, info = run_gpu(cfg, steps, kernel="per_step", level0=level0)
            ref = run_oracle(oracle, cfg, steps, level0=level0)
            assert info["kernel"] == "per_step" and info["launches"] == steps
            assert rel_err_rows(got, ref, cfg) <= TOL[dtype], (n, level0, steps)


@pytest.mark.parametrize("dtype", ["f64", "f32"])
def test_step_1d_entry_point_matches_run(oracle, dtype):
    cfg = inputs.random_rods(2, 516, dtype, seed=5)
    a, _ = run_gpu(cfg, 7, kernel="per_step", via="step")
    b, _ = run_gpu(cfg, 7, kernel="per_step", via="run")
    np.testing.assert_array_equal(a, b)
    assert rel_err_rows(a, run_oracle(oracle, cfg, 7)) <= TOL[dtype]


def test_unaligned_pointers_take_the_scalar_kernel(oracle):
    import torch
    from paper_1310_3422_b200 import libge
    cfg = inputs.random_rods(1, 1000, "f64", seed=9)
    dev = torch.device("cuda:0")
    buf = torch.zeros(1000 + 1, dtype=torch.float64, device=dev)
    out = torch.zeros(1000 + 1, dtype=torch.float64, device=dev)
    u, v = buf[1:], out[1:]                       # 8-byte aligned, not 16
    u.copy_(torch.from_numpy(cfg["u0"].reshape(-1)))
    s = torch.cuda.current_stream(dev).cuda_stream
    with libge.Plan(cfg, kernel="per_step", stream=s) as plan:
        plan.step(u.data_ptr(), v.data_ptr(), s)
        plan.step(v.data_ptr(), u.data_ptr(), s)
        torch.cuda.synchronize()
    assert rel_err(u.cpu().numpy(), run_oracle(oracle, cfg, 2).reshape(-1)) <= 1e-14


def test_step_rejects_bad_arguments():
    import torch
    from paper_1310_3422_b200 import libge
    cfg = inputs.random_rods(1, 64, "f64")
    u = torch.zeros(128, dtype=torch.float64, device="cuda:0")
    with libge.Plan(cfg) as plan:
        for a, b in ((u.data_ptr(), u.data_ptr()), (0, u.data_ptr()), (u.data_ptr(), u.data_ptr() + 8 * 32),
                     (u.data_ptr() + 4, u.data_ptr() + 8 * 64)):
            with pytest.raises(libge.GeError) as ei:
                plan.step(a, b)
            assert ei.value.status == libge.GE_EINVAL
        with pytest.raises(libge.GeError):
            libge.ge_step_2d(plan.handle, u.data_ptr(), u.data_ptr() + 8 * 64)
        with pytest.raises(libge.GeError):
            plan.run(u.data_ptr(), -1)
        plan.run(u.data_ptr(), 0)
        assert plan.level == 0 and plan.info()["launches"] == 0


# ------------------------------------------------------------------ strategy B, 1-D ------
@pytest.mark.parametrize("dtype,tb,tc", [("f64", 0, 0), ("f64", 1, 8), ("f64", 2, 16), ("f64", 7, 8), ("f64", 13, 16),
                                         ("f64", 32, 8), ("f64", 100, 16), ("f64", 24, 32), ("f64", 16, 18), ("f64", 7, 18), ("f64", 61, 18), ("f64", 20, 22), ("f64", 9, 26), ("f32", 0, 0), ("f32", 50, 64),
                                         ("f32", 16, 36), ("f32", 9, 36), ("f32", 120, 36), ("f32", 20, 44), ("f32", 33, 52), ("f32", 1, 32), ("f32", 3, 16),
                                         ("f32", 6, 32), ("f32", 8, 16), ("f32", 21, 32), ("f32", 40, 16), ("f32", 200, 32)])
@pytest.mark.parametrize("n", [8, 224, 232, 2048, 10000, 3 * 4096 + 8])
def test_temporal_1d(oracle, dtype, tb, tc, n):
    """Strategy B against the oracle: every starting phase, odd and even block lengths (pre/post
    realignment shifts), tiles with both ghosts, ragged last tile; the warp-per-tile kernels (generic
    and drift-free) and the TMA-staged persistent kernel (tc = 18, 22, 26 / 36, 44, 52)."""
    if tc in (18, 22, 26, 36, 44, 52) and n < 32 * tc:
        pytest.skip("the TMA-staged kernel needs a rod of at least one tile")
    cfg = inputs.random_rods(2, n, dtype, seed=7 * n + tb)
    for level0, steps in ((0, 1), (1, 16), (0, 40), (1, 37), (0, 101)):
        got, info = run_gpu(cfg, steps, kernel="temporal", tb=tb, level0=level0, tc=tc)
        ref = run_oracle(oracle, cfg, steps, level0=level0)
        assert info["kernel"] == "temporal"
        if steps >= 40 and tb != 1:
            assert info["launches"] < steps        # the blocked kernel really ran
        assert rel_err_rows(got, ref, cfg) <= TOL[dtype], (n, level0, steps, info)


def test_temporal_1d_bitwise_equals_per_step():
    """The blocked kernel evaluates the same factored form in the same order as the per-level kernel:
    results are bit-identical, whatever tb, C and the starting phase."""
    for dtype in ("f64", "f32"):
        cfg = inputs.random_rods(3, 6000, dtype, seed=11)
        for level0 in (0, 1):
            a, _ = run_gpu(cfg, 57, kernel="per_step", level0=level0)
            for tb, tc in ((16, 0), (5, 0), (57, 0), (20, 8 if dtype == "f64" else 16), (33, 32 if dtype == "f64" else 64),
                           (16, 18 if dtype == "f64" else 36), (23, 18 if dtype == "f64" else 36)):
                b, info = run_gpu(cfg, 57, kernel="temporal", tb=tb, level0=level0, tc=tc)
                np.testing.assert_array_equal(a, b, err_msg=str((dtype, level0, tb, tc, info)))


@pytest.mark.parametrize("dtype", ["f64", "f32"])
def test_temporal_1d_odd_n_batched_stays_blocked(oracle, dtype):
    """Batched rods of odd length start at alternating alignments: no vector kernel, but still tb levels per launch
    (the unaligned form of the warp-per-tile kernel; r01 fell back to one launch per level here)."""
    cfg = inputs.random_rods(2, 1001, dtype, seed=77)
    got, info = run_gpu(cfg, 33, kernel="temporal")
    assert info["launches"] <= 3, info
    assert rel_err_rows(got, run_oracle(oracle, cfg, 33)) <= TOL[dtype]
    same, _ = run_gpu(cfg, 33, kernel="per_step")
    np.testing.assert_array_equal(got, same)


@pytest.mark.parametrize("dtype", ["f64", "f32"])
@pytest.mark.parametrize("n", [1001, 1002, 4099, 2 ** 20 + 1, 2 ** 20 + 2, 2 ** 20 + 3])
@pytest.mark.parametrize("kernel", ["temporal", "auto", "persistent"])
def test_awkward_lengths_stay_on_the_blocked_kernels(oracle, dtype, n, kernel):
    """A single rod whose length is odd (a first-class case of the scheme: the last node is alone in phase 0,
    paired in phase 1) or not a multiple of the 16-byte vector: the blocked kernel marches the prefix, the
    end-piece kernel (ge_tail.cuh) recomputes the last 2 tb + 2 + nx % V nodes from the true boundary -- no
    silent fall to one launch per level.  Both starting phases, odd level counts; against the oracle and bit
    for bit against the per-level kernel."""
    cfg = inputs.random_rods(1, n, dtype, seed=n % 977)
    v = 2 if dtype == "f64" else 4
    for level0, steps in ((0, 1), (1, 40), (0, 101)):
        got, info = run_gpu(cfg, steps, kernel=kernel, level0=level0)
        ref = run_oracle(oracle, cfg, steps, level0=level0)
        assert rel_err_rows(got, ref, cfg) <= TOL[dtype], (n, level0, steps, info)
        if n % v and steps >= 40 and info["resident_path"] == 0:
            assert info["launches"] < steps, info            # blocked launches + one end piece each
        same, _ = run_gpu(cfg, steps, kernel="per_step", level0=level0)
        np.testing.assert_array_equal(got, same, err_msg=str((dtype, n, kernel, level0, steps, info)))


@pytest.mark.parametrize("dtype", ["f64", "f32"])
@pytest.mark.parametrize("batch,n", [(7, 1001), (5, 4098), (3, 4097), (40, 99), (33, 100), (2, 40001), (9, 515), (4, 31)])
def test_batched_rods_of_awkward_lengths_stay_blocked(oracle, dtype, batch, n):
    """Batched rods whose length is not a multiple of the 16-byte vector start at unaligned addresses: the
    warp-per-tile kernel reads and writes them with coalesced scalar accesses transposed through shared memory
    (ge_temporal.cuh, UA) instead of falling to one launch per level.  Per-rod r and boundary values, both starting
    phases, odd level counts; against the oracle and bit for bit against the per-level kernel."""
    cfg = inputs.random_rods(batch, n, dtype, seed=batch * 1000 + n, r_hi=4.0)
    v = 2 if dtype == "f64" else 4
    for level0, steps in ((0, 1), (1, 40), (0, 101), (1, 23)):
        got, info = run_gpu(cfg, steps, kernel="temporal", level0=level0)
        ref = run_oracle(oracle, cfg, steps, level0=level0)
        assert rel_err_rows(got, ref, cfg) <= TOL[dtype], (batch, n, level0, steps, info)
        if n % v and steps >= 23:
            assert info["launches"] <= steps // 8 + 2, info
        same, _ = run_gpu(cfg, steps, kernel="per_step", level0=level0)
        np.testing.assert_array_equal(got, same, err_msg=str((dtype, batch, n, level0, steps, info)))
        auto, _ = run_gpu(cfg, steps, level0=level0)
        np.testing.assert_array_equal(auto, same)


@pytest.mark.parametrize("dtype", ["f64", "f32"])
@pytest.mark.parametrize("batch,n,off", [(1, 2 ** 16, 1), (1, 4099, 1), (6, 2048, 1), (3, 1000, 3), (1, 2 ** 20, 2)])
def test_unaligned_pointers_stay_blocked(oracle, dtype, batch, n, off):
    """A state that starts `off` elements after a 16-byte boundary (a slice of a larger buffer): ge_run must neither
    fault nor fall to one launch per level."""
    import torch
    from paper_1310_3422_b200 import libge
    cfg = inputs.random_rods(batch, n, dtype, seed=n % 991 + off)
    dev = torch.device("cuda:0")
    stream = torch.cuda.current_stream(dev).cuda_stream
    big = torch.zeros(batch * n + 8, dtype=torch.float64 if dtype == "f64" else torch.float32, device=dev)
    es = big.element_size()
    if off * es % 16 == 0:
        pytest.skip("this offset is 16-byte aligned for the dtype")
    u = big[off:off + batch * n]
    u.copy_(torch.from_numpy(cfg["u0"].reshape(-1)).to(dev))
    assert u.data_ptr() % 16 != 0
    steps = 61
    with libge.Plan(cfg, kernel="temporal", stream=stream) as plan:
        plan.run(u.data_ptr(), steps, stream)
        torch.cuda.synchronize(dev)
        info = plan.info()
    got = u.cpu().numpy().reshape(cfg["u0"].shape)
    assert info["launches"] <= steps // 8 + 2, info
    assert float(big[:off].abs().max()) == 0.0 and float(big[off + batch * n:].abs().max()) == 0.0   # nothing outside
    same, _ = run_gpu(cfg, steps, kernel="per_step")
    np.testing.assert_array_equal(got, same)
    ref = run_oracle(oracle, cfg, steps)
    assert rel_err_rows(got, ref, cfg) <= TOL[dtype]


@pytest.mark.parametrize("dtype", ["f64", "f32"])
def test_blocked_1d_runs_take_an_even_number_of_launches(oracle, dtype):
    """The state ping-pongs between the caller's buffer and the plan's scratch level; ge_run picks the block length
    so that runs of three or more launches end in the caller's buffer (no copy of the whole state).  Results do not
    depend on the split: bit for bit the per-level kernel's."""
    for batch, n in ((1, 2 ** 17), (3, 8192), (2, 4097)):
        cfg = inputs.random_rods(batch, n, dtype, seed=n % 97)
        for level0, steps in ((0, 100), (1, 100), (0, 220), (1, 61), (0, 59), (0, 300)):
            got, info = run_gpu(cfg, steps, kernel="temporal", tb=20, level0=level0)
            assert info["kernel"] == "temporal" and info["launches"] % 2 == 0 and info["launches"] <= steps // 8 + 2, (batch, n, level0, steps, info)
            same, _ = run_gpu(cfg, steps, kernel="per_step", level0=level0)
            np.testing.assert_array_equal(got, same, err_msg=str((dtype, batch, n, level0, steps, info)))
    ref = run_oracle(oracle, cfg, 300)
    assert rel_err_rows(got, ref, cfg) <= TOL[dtype]


def test_run_is_deterministic():
    cfg = inputs.random_rods(4, 4096, "f32", seed=3)
    a, _ = run_gpu(cfg, 100)
    b, _ = run_gpu(cfg, 100)
    np.testing.assert_array_equal(a, b)


def test_run_host_matches_run(oracle):
    cfg = inputs.random_rods(3, 2048, "f64", seed=31)
    a, _ = run_gpu(cfg, 50, via="host")
    b, _ = run_gpu(cfg, 50, via="run")
    np.testing.assert_array_equal(a, b)


# ------------------------------------------------------------------ strategy C, 1-D ------
@pytest.mark.parametrize("dtype,n,rc", [("f32", 64, 0), ("f32", 512, 16), ("f32", 4096, 0), ("f32", 4096, 64),
                                        ("f32", 4096, 32), ("f32", 2048 + 128, 0), ("f32", 96, 0), ("f32", 16384, 0),
                                        ("f64", 8, 0), ("f64", 64, 0), ("f64", 2048, 0), ("f64", 2048, 32),
                                        ("f64", 2048, 16), ("f64", 1000, 8), ("f64", 16384, 64),
                                        # short rods on the small lane widths (C = 4, 8 fp32 / 2, 4 fp64)
                                        ("f32", 4, 0), ("f32", 8, 0), ("f32", 100, 0), ("f32", 100, 4), ("f32", 1000, 0), ("f32", 1000, 8),
                                        ("f32", 1016, 0), ("f64", 2, 0), ("f64", 4, 0), ("f64", 6, 0), ("f64", 50, 0), ("f64", 100, 4),
                                        ("f64", 62, 2), ("f64", 500, 2), ("f64", 510, 0)])
def test_persistent_rods(oracle, dtype, n, rc):
    """Strategy C, path 1 (a rod per CTA, state in registers for the whole run): one launch whatever
    the number of levels; one warp (shuffles only) and several warps (shared-memory edge exchange);
    lanes and warps that hold no nodes; both starting phases, odd and even level counts; per-rod r
    and unequal boundary values.  Must equal the per-level kernel bit for bit."""
    cfg = inputs.random_rods(5, n, dtype, seed=3 * n + rc)
    for level0, steps in ((0, 1), (1, 1), (0, 2), (1, 2), (0, 37), (1, 64), (0, 301)):
        got, info = run_gpu(cfg, steps, kernel="persistent", level0=level0, rc=rc)
        assert info["kernel"] == "persistent" and info["resident_path"] == 1 and info["launches"] == 1, info
        if rc:
            assert info["resident_c"] == rc
        ref = run_oracle(oracle, cfg, steps, level0=level0)
        assert rel_err_rows(got, ref, cfg) <= TOL[dtype], (n, level0, steps, info)
        same, _ = run_gpu(cfg, steps, kernel="per_step", level0=level0)
        np.testing.assert_array_equal(got, same, err_msg=str((dtype, n, level0, steps, info)))


@pytest.mark.parametrize("dtype,n,rc,hl,rtb,sync", [
    ("f64", 4096, 0, 0, 0, 2), ("f64", 4096, 16, 1, 0, None), ("f64", 30720, 0, 1, 6, 2),
    ("f64", 100000, 0, 2, 0, None), ("f64", 100000, 16, 3, 10, 1), ("f64", 2 ** 20, 0, 0, 0, None),
    ("f64", 2 ** 20, 0, 0, 0, 1), ("f64", 2 ** 20, 0, 0, 0, 0), ("f64", 30720, 0, 2, 4, 0),
    ("f32", 16384 * 4, 0, 0, 0, 2), ("f32", 16384 * 4, 0, 1, 8, 0), ("f32", 2 ** 20, 128, 1, 0, 2), ("f32", 200000 - 200000 % 64, 32, 2, 20, None),
    ("f32", 2 ** 20, 0, 0, 0, 1),
    ("f64", 2 ** 20, 0, 0, 0, 3), ("f64", 30720, 0, 1, 8, 3), ("f64", 100000, 16, 3, 10, 3), ("f32", 16384 * 4, 0, 0, 0, 3),
    ("f32", 2 ** 20, 128, 1, 0, 3),
    # thread-block clusters of 2 / 4 / 8 / 16 CTAs (sync = 4 .. 7)
    ("f64", 2 ** 20, 0, 0, 0, 4), ("f64", 2 ** 20, 0, 0, 0, 5), ("f64", 2 ** 20, 0, 0, 0, 6), ("f64", 2 ** 20, 0, 0, 0, 7),
    ("f64", 30720, 0, 1, 6, 6), ("f64", 100000, 16, 3, 10, 5), ("f64", 4096, 0, 0, 0, 6), ("f32", 16384 * 4, 0, 1, 8, 6),
    ("f32", 2 ** 20, 128, 1, 0, 4), ("f32", 2 ** 20, 0, 0, 0, 7)])
def test_persistent_whole_chip(oracle, dtype, n, rc, hl, rtb, sync):
    """Strategy C, path 2 (one rod spread over the chip by a cooperative launch, tiles meet every tb
    levels): grid-wide barrier (default), neighbour flags (sync=0), flag-in-data lines (sync=2) and
    staggered flag-in-data lines (sync=3: published every tb/2 levels, consumed every other time), thread-block
    clusters (sync=4..7: shared memory / DSMEM + the cluster barrier inside a cluster, flags between clusters), one
    and several halo lanes, many meetings, no
    meeting, ragged last tile, both starting phases, odd level counts, and several ge_run calls on
    one plan (the flag epoch carries over).  Must equal the per-level kernel bit for bit."""
    from paper_1310_3422_b200 import libge
    cfg = inputs.random_rods(1, n, dtype, seed=n % 1000 + rc + hl)
    for level0, steps, chunks in ((0, 1, None), (1, 2, None), (0, 40, None), (1, 77, None), (0, 203, (100, 3, 100))):
        try:
            got, info = run_gpu(cfg, steps, kernel="persistent", level0=level0, rc=rc, hl=hl, rtb=rtb, sync=sync,
                                chunks=chunks)
        except libge.GeError as e:
            if sync is not None and sync >= 4 and e.status == libge.GE_EINVAL:
                pytest.skip("the rod cannot stay resident with clusters of this size")
            raise
        assert info["kernel"] == "persistent" and info["resident_path"] == 2, info
        assert info["launches"] == (len(chunks) if chunks else 1)
        assert info["resident_warps"] <= info["resident_capacity"]
        if steps > 2 * info["resident_tb"]:
            assert info["meetings"] >= steps // info["resident_tb"] - 3
        same, _ = run_gpu(cfg, steps, kernel="per_step", level0=level0)
        np.testing.assert_array_equal(got, same, err_msg=str((dtype, n, level0, steps, info)))
    ref = run_oracle(oracle, cfg, 77, level0=1)
    got, _ = run_gpu(cfg, 77, kernel="persistent", level0=1, rc=rc, hl=hl, rtb=rtb, sync=sync)
    assert rel_err_rows(got, ref, cfg) <= TOL[dtype]


def test_persistent_falls_back_when_the_shape_does_not_fit(oracle):
    # odd N, batched: no resident kernel, no vector kernel either -> the unaligned blocked kernel
    cfg = inputs.random_rods(2, 1001, "f64", seed=5)
    got, info = run_gpu(cfg, 20, kernel="persistent")
    assert info["kernel"] == "temporal" and info["resident_path"] == 0 and info["launches"] <= 2
    assert rel_err_rows(got, run_oracle(oracle, cfg, 20), cfg) <= TOL["f64"]
    # 2-D: strategy C is 1-D only
    cfg = inputs.random_grid(64, 64, "f32", seed=6)
    got, info = run_gpu(cfg, 16, kernel="persistent")
    assert info["kernel"] == "temporal" and info["resident_path"] == 0
    assert rel_err(got, run_oracle(oracle, cfg, 16)) <= TOL["f32"]
    # batched rods too long for a CTA
    cfg = inputs.random_rods(2, 128 * 32 * 8 * 2, "f32", seed=7)
    got, info = run_gpu(cfg, 33, kernel="persistent")
    assert info["kernel"] == "temporal" and info["launches"] < 33
    assert rel_err_rows(got, run_oracle(oracle, cfg, 33), cfg) <= TOL["f32"]


def test_auto_picks_the_resident_kernels_when_the_state_fits_on_chip():
    for cfg, path in ((inputs.make_c1(), 1), (inputs.make_c3(batch=4, n=4096, steps=10), 1),
                      (inputs.make_c2(n=2 ** 20, steps=10), 2), (inputs.make_c4(n=2 ** 24, steps=10), 0)):
        _, info = run_gpu(cfg, 10)
        assert info["resident_path"] == path, (cfg["name"], info)
        assert info["kernel"] == ("persistent" if path else "temporal")


# ------------------------------------------------------------------ sub-domain length k >= 2 ------
@pytest.mark.parametrize("dtype", ["f64", "f32"])
@pytest.mark.parametrize("k,n", [(2, 1), (2, 2), (2, 3), (2, 6), (2, 7), (3, 10), (3, 64), (5, 1003), (16, 62), (16, 30),
                                 (16, 8206), (16, 5000), (7, 4099), (64, 20000), (100, 150), (1000, 5000)])
def test_general_k_per_level(oracle, dtype, k, n):
    """The paper's general scheme: confluence pairs every 2k
    nodes joined by Saul'yev sweeps.  Paper-shaped layouts ((N+2) mod 2k == 0, e.g. k = 16,
    N = 8206 -- the paper's "8208" nodes), ragged ones, rods shorter than a sub-domain, both starting
    phases, per-rod r and unequal boundary values."""
    cfg = inputs.random_rods(3, n, dtype, seed=17 * k + n)
    for level0, steps in ((0, 1), (1, 1), (0, 2), (1, 7), (0, 40)):
        got, info = run_gpu(cfg, steps, level0=level0, k=k, kernel="per_step")
        ref = run_oracle(oracle, cfg, steps, level0=level0, k=k)
        assert info["kernel"] == "per_step" and info["launches"] == steps
        assert rel_err_rows(got, ref, cfg) <= TOL[dtype], (k, n, level0, steps)
        # strategy C (the rod resident in shared memory, one launch): AUTO picks it when the rod fits
        res, info = run_gpu(cfg, steps, level0=level0, k=k)
        assert info["kernel"] == "persistent" and info["resident_path"] == 3 and info["launches"] == 1, info
        np.testing.assert_array_equal(res, got)


@pytest.mark.parametrize("dtype", ["f64", "f32"])
@pytest.mark.parametrize("k,n,tb", [(2, 40000, 8), (3, 50001, 8), (16, 100000, 8), (16, 2 ** 18 - 2, 16), (64, 200000, 4),
                                    (5, 30011, 13), (16, 70000, 1)])
def test_general_k_temporal(oracle, dtype, k, n, tb):
    """Strategy B for k >= 2 (ge1d_temporal_k_kernel): tb levels per launch on tiles whose window carries
    tb (k+1) + 2k + 2 nodes of halo per cut side; several tiles, ragged last tile, rod ends inside a window, both
    starting phases, >= 200 levels, a level count that is not a multiple of tb.  Against the oracle and bit
    for bit against the per-level kernel."""
    cfg = inputs.random_rods(2, n, dtype, seed=13 * k + n % 1000)
    for level0, steps in ((0, 1), (1, 2 * tb + 3), (0, 203)):
        got, info = run_gpu(cfg, steps, level0=level0, k=k, kernel="temporal", tb=tb, kform=0)
        assert info["kernel"] == "temporal" and info["tb"] == tb, info
        assert info["launches"] == -(-steps // tb), info
        ref = run_oracle(oracle, cfg, steps, level0=level0, k=k)
        assert rel_err_rows(got, ref, cfg) <= TOL[dtype], (k, n, level0, steps, info)
        same, i2 = run_gpu(cfg, steps, level0=level0, k=k, kernel="per_step")
        assert i2["launches"] == steps
        np.testing.assert_array_equal(got, same, err_msg=str((k, n, level0, steps)))


@pytest.mark.parametrize("dtype", ["f64", "f32"])
@pytest.mark.parametrize("k,n,tb,batch", [(2, 40000, 8, 1), (4, 100000, 16, 1), (8, 70001, 8, 1), (16, 2 ** 18 - 2, 16, 1),
                                          (16, 100003, 5, 1), (16, 40000, 8, 3), (32, 200000, 8, 1), (16, 2 ** 20, 16, 1)])
def test_general_k_register_units(oracle, dtype, k, n, tb, batch):
    """The register-resident form of strategy B for k >= 2 (ge1d_unit_k_kernel: a thread holds 2k nodes for tb
    levels, one value crosses a lane boundary per level) + the shared-memory kernel on the two ends of the rod:
    several tiles, ragged and odd lengths, batched rods, both starting phases, odd level counts.  Against the
    oracle and bit for bit against the per-level kernel and the shared-memory form."""
    if k == 32 and dtype == "f64":
        pytest.skip("k = 32 is compiled for fp32 only")
    cfg = inputs.random_rods(batch, n, dtype, seed=7 * k + n % 1000)
    for level0, steps in ((0, 1), (1, 2 * tb + 3), (0, 203)):
        got, info = run_gpu(cfg, steps, level0=level0, k=k, kernel="temporal", tb=tb, kform=1)
        assert info["kernel"] == "temporal" and info["launches"] == 2 * -(-steps // tb), info   # unit kernel + end windows
        ref = run_oracle(oracle, cfg, steps, level0=level0, k=k)
        assert rel_err_rows(got, ref, cfg) <= TOL[dtype], (k, n, level0, steps, info)
        same, _ = run_gpu(cfg, steps, level0=level0, k=k, kernel="per_step")
        np.testing.assert_array_equal(got, same, err_msg=str((k, n, level0, steps)))
        smem, i3 = run_gpu(cfg, steps, level0=level0, k=k, kernel="temporal", tb=tb, kform=0)
        assert i3["launches"] == -(-steps // tb)
        np.testing.assert_array_equal(got, smem)


def test_general_k_auto_takes_the_blocked_kernel_on_long_rods():
    cfg = inputs.random_rods(1, 2 ** 20 - 2, "f64", seed=4)
    _, info = run_gpu(cfg, 96, k=16, kform=0)
    assert info["kernel"] == "temporal" and info["tb"] == 32 and info["launches"] == 3, info
    assert info["tile_loaded"] - info["tile_valid"] == 2 * (32 * 17 + 2 * 16 + 2)
    _, info = run_gpu(cfg, 96, k=16)
    assert info["kernel"] == "temporal" and info["launches"] == 6, info        # register units + end windows
    _, info = run_gpu(inputs.random_rods(1, 2 ** 20 - 2, "f64", seed=4), 48, k=3)
    assert info["kernel"] == "temporal" and info["tb"] == 16 and info["launches"] == 3, info   # k = 3: shared-memory form


def test_general_k_resident_needs_the_rod_to_fit():
    cfg = inputs.random_rods(1, 100000, "f64", seed=1)           # 800 KB: more than a CTA's shared memory
    _, info = run_gpu(cfg, 3, k=16)
    assert info["kernel"] == "temporal" and info["resident_path"] == 0 and info["launches"] == 2
    _, info = run_gpu(cfg, 3, k=16, kernel="per_step")
    assert info["kernel"] == "per_step" and info["launches"] == 3
    cfg = inputs.random_rods(1, 40000, "f32", seed=1)            # fits, but 10 001 units > 1024 threads at k = 2
    _, info = run_gpu(cfg, 3, k=2)
    assert info["kernel"] == "temporal"


def test_general_k_plan_rejects_the_two_point_resident_tuning(oracle):
    """GE_TUNE_RESIDENT_C configures the register-resident kernels, which are the k = 1 scheme: a k >= 2 plan
    on its shared-memory resident path must refuse it (and keep computing the k = 16 scheme)."""
    import torch
    from paper_1310_3422_b200 import libge
    cfg = inputs.random_rods(2, 8192 - 2, "f64", seed=3)
    u = torch.from_numpy(cfg["u0"]).to("cuda:0")
    with libge.Plan(cfg, group_k=16, kernel="persistent") as plan:
        assert plan.info()["resident_path"] == 3
        for c in (8, 16, 32, 64):
            with pytest.raises(libge.GeError) as ei:
                plan.tune(libge.GE_TUNE_RESIDENT_C, c)
            assert ei.value.status == libge.GE_EUNSUPPORTED
        assert plan.info()["resident_path"] == 3
        plan.run(u.data_ptr(), 30)
        torch.cuda.synchronize()
    ref = run_oracle(oracle, cfg, 30, k=16)
    assert rel_err_rows(u.cpu().numpy(), ref, cfg) <= TOL["f64"]


def test_general_k_matches_the_closed_form(oracle):
    """k = 16 on N = 254 (the paper's SDC width 32): the end state follows e^{-pi^2 t} sin(pi x) to the
    oracle's own error (tests/golden P6: 5.35e-5 at t ~ 0.1, r = 1)."""
    n, r = 254, 1.0
    x = np.arange(1, n + 1) / (n + 1.0)
    steps = int(round(0.1 * (n + 1) ** 2 / r))
    cfg = dict(inputs.random_rods(1, n, "f64"), r=np.array([r]), bc_lo=np.array([0.0]), bc_hi=np.array([0.0]),
               u0=np.sin(np.pi * x)[None, :].copy())
    got, _ = run_gpu(cfg, steps, k=16)
    ref = run_oracle(oracle, cfg, steps, k=16)
    assert rel_err_rows(got, ref, cfg) <= TOL["f64"]
    t = steps * r / (n + 1.0) ** 2
    err = np.abs(got.reshape(-1) - np.exp(-np.pi ** 2 * t) * np.sin(np.pi * x)).max()
    assert 3e-5 < err < 8e-5, err


# ------------------------------------------------------------------ 2-D ------
@pytest.mark.parametrize("dtype", ["f64", "f32"])
@pytest.mark.parametrize("nx,ny", [(1, 1), (2, 2), (3, 3), (4, 4), (5, 4), (4, 7), (8, 8), (64, 32), (130, 67), (131, 66), (256, 256)])
def test_per_step_2d(oracle, dtype, nx, ny):
    cfg = inputs.random_grid(nx, ny, dtype, seed=nx * 1000 + ny, r=1.7)
    for level0 in (0, 1):
        for steps in (1, 2, 5):
            got, info = run_gpu(cfg, steps, level0=level0)
            ref = run_oracle(oracle, cfg, steps, level0=level0)
            assert info["launches"] == steps
            assert rel_err(got, ref) <= (2e-14 if dtype == "f64" else 3e-6), (nx, ny, level0, steps)


def _launches_2d(nx, tb, level0, steps, dtype):
    """ge_run's 2-D schedule: the strip kernel (nx % 4 == 0, nx >= one strip: 128 columns in fp32, 64 in
    fp64) starts at odd levels only."""
    strips = nx % 4 == 0 and nx >= (128 if dtype == "f32" else 64)
    level, left, n = level0, steps, 0
    while left > 0:
        if strips and left > tb and level % 2 == 0:
            d = 1
        elif strips and left >= tb and level % 2 == 1:
            d = tb
        elif not strips and left >= tb:
            d = tb
        else:
            d = 1
        level += d; left -= d; n += 1
    return n


@pytest.mark.parametrize("dtype", ["f64", "f32"])
@pytest.mark.parametrize("nx,ny,tb,hp", [(8, 8, 4, 64), (64, 32, 8, 4), (256, 256, 8, 64), (232, 70, 4, 8),
                                         (500, 301, 8, 16), (1024, 96, 8, 64), (116, 1000, 4, 100),
                                         (128, 16, 4, 2), (128, 130, 6, 5), (352, 77, 6, 64), (240, 64, 8, 3),
                                         (1000, 37, 4, 64), (2048, 20, 8, 64)])
def test_temporal_2d(oracle, dtype, nx, ny, tb, hp):
    """Strategy B in 2-D (warp strips streaming along y): the drift-free strip kernel (nx >= 128 in fp32, 64 in fp64:
    aligned first/last strips, R/L stages, x-edge groups on lane 0 / 31, y-edge groups in the
    generic stage) and the drifting kernel for narrow grids; several strips and segments, ragged
    last strip/segment, odd ny, both starting phases, and a remainder of levels that falls back to
    the per-level kernel.  Must equal the per-level kernel bit for bit."""
    cfg = inputs.random_grid(nx, ny, dtype, seed=nx * 7 + ny, r=1.7)
    for level0, steps in ((0, tb), (1, tb), (0, 2 * tb + 3), (1, 3 * tb), (0, 4 * tb + 1)):
        got, info = run_gpu(cfg, steps, kernel="temporal", tb=tb, level0=level0, hp=hp)
        ref = run_oracle(oracle, cfg, steps, level0=level0)
        assert info["kernel"] == "temporal" and info["launches"] == _launches_2d(nx, tb, level0, steps, dtype), info
        assert rel_err(got, ref) <= (1e-13 if dtype == "f64" else 1e-5), (nx, ny, level0, steps, info)
        same, _ = run_gpu(cfg, steps, kernel="per_step", level0=level0)
        np.testing.assert_array_equal(got, same, err_msg=str((nx, ny, level0, steps)))


@pytest.mark.parametrize("dtype", ["f64", "f32"])
@pytest.mark.parametrize("coop", [2, 4, 8])
@pytest.mark.parametrize("nx,ny,hp", [(1024, 64, 8), (1032, 77, 5), (2048, 40, 64), (2600, 130, 11), (4096 + 8, 33, 3)])
def test_temporal_2d_cooperative_strips(oracle, dtype, coop, nx, ny, hp):
    """The cooperative form of the strip kernel (GE_TUNE_STRIP_COOP: 4 or 8 warps of a CTA share one strip and
    pass their edge right-hand sides through shared memory behind pairwise named barriers): one strip and
    several, ragged last strip, segments shorter than the pipeline, x- and y-edge groups (the CTA-wide slow
    path), both starting phases.  Must equal the per-level kernel bit for bit and match the oracle."""
    cfg = inputs.random_grid(nx, ny, dtype, seed=nx + 3 * ny, r=1.7)
    tb = 6
    for level0, steps in ((1, tb), (0, 2 * tb + 3), (1, 5 * tb)):
        got, info = run_gpu(cfg, steps, kernel="temporal", tb=tb, level0=level0, hp=hp, coop=coop)
        assert info["kernel"] == "temporal" and info["launches"] == _launches_2d(nx, tb, level0, steps, dtype), info
        assert info["tile_loaded"] == coop * (128 if dtype == "f32" else 64)
        ref = run_oracle(oracle, cfg, steps, level0=level0)
        assert rel_err(got, ref) <= (1e-13 if dtype == "f64" else 1e-5), (nx, ny, level0, steps, info)
        same, _ = run_gpu(cfg, steps, kernel="per_step", level0=level0)
        np.testing.assert_array_equal(got, same, err_msg=str((nx, ny, coop, level0, steps)))


def test_step_2d_entry_point(oracle):
    cfg = inputs.random_grid(96, 40, "f64", seed=8)
    a, _ = run_gpu(cfg, 4, via="step")
    assert rel_err(a, run_oracle(oracle, cfg, 4)) <= 1e-14


# ------------------------------------------------------------------ BASELINE configs ------
def test_config1_exact(oracle):
    cfg = inputs.make_c1()
    ref = run_oracle(oracle, cfg, cfg["steps"])
    for kernel in ("per_step", "temporal"):
        got, _ = run_gpu(cfg, cfg["steps"], kernel=kernel)
        assert rel_err(got, ref) <= TOL["f64"]
    x = np.arange(1, 65) / 65.0
    exact = np.exp(-np.pi ** 2 * 1000 / 65.0 ** 2) * np.sin(np.pi * x)
    assert abs(np.abs(got.reshape(-1) - exact).max() - 4.6957e-4) < 1e-7     # tests/golden P7


def test_config2_reduced(oracle):
    cfg = inputs.make_c2(n=2 ** 14, steps=10000)
    ref = run_oracle(oracle, cfg, cfg["steps"])
    for kernel in ("per_step", "temporal"):
        got, _ = run_gpu(cfg, cfg["steps"], kernel=kernel)
        assert rel_err(got, ref) <= TOL["f64"], kernel


def test_config3_reduced(oracle):
    cfg = inputs.make_c3(batch=48, n=4096, steps=2000)
    ref = run_oracle(oracle, cfg, cfg["steps"])
    for kernel in ("per_step", "auto"):
        got, _ = run_gpu(cfg, cfg["steps"], kernel=kernel)
        assert rel_err_rows(got, ref) <= TOL["f32"], kernel


def test_config4_reduced(oracle):
    cfg = inputs.make_c4(n=2 ** 20, steps=200)
    ref = run_oracle(oracle, cfg, cfg["steps"])
    for kernel in ("per_step", "temporal"):
        got, _ = run_gpu(cfg, cfg["steps"], kernel=kernel)
        assert rel_err(got, ref) <= TOL["f64"], kernel


@pytest.mark.parametrize("dtype", ["f32", "f64"])
def test_config5_reduced(oracle, dtype):
    cfg = inputs.make_c5(n=512, steps=1000, dtype=dtype)
    ref = run_oracle(oracle, cfg, cfg["steps"])
    for kernel in ("per_step", "temporal"):
        got, _ = run_gpu(cfg, cfg["steps"], kernel=kernel)
        assert rel_err(got, ref) <= TOL[dtype], kernel
