#!/usr/bin/env python
"""bench.py -- grid-point updates/s of the GE time-marching loop (arXiv 1310.3422) on B200.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--config c4|c2|c3|c5_f32|c5_f64]
                    [--kernel auto|per_step|temporal|persistent] [--tb T] [--impl ours|reference]

One "step" = one pass of the whole hot path over one synthetic grid: one
`ge_run` of the config's full number of levels.  Default workload: BASELINE.json configs[3] (C4,
N = 2^28 fp64, r = 2, 200 levels) -- the largest 1-D grid, the one the metric's "achieved HBM GB/s
on the largest grids" is quoted on; the state (2 GiB) is larger than L2, so no flush is needed
between timed iterations.  Rank 0 prints ONE JSON line (DESIGN.md "Measurement" explains every key).

N > 1 (torchrun): "replicas only" -- every rank marches its own copy of the workload, no data-path
collective; value = updates of all ranks / max-over-ranks device time.

--impl reference times the ORACLE (oracle/ge_ref.c, plain fp64 C, one host core) on a bounded sample
of the same workload; it is a deliberately slow baseline, not the target.

Beside the contract's keys the default line carries: `alu_peaks` (FFMA / DFMA throughput measured in this
run by libge's ge_fma_probe, the denominator of every "bound": "alu" roofline), `parity` (sampled
dependency cones of a run from the config's initial state against the oracle), `cpu_baseline` with a
one-thread and an all-cores leg on ONE sample (the same one --impl reference times), `secondary` (C5 f32,
C5 f64, C2, C3 and the 3-D boxes device-resident, so that the 2-D half of the north_star target and the 3-D
row are in the driver's record),
and the PCIe ceiling beside `e2e`.  `--sweep sync` is the synchronisation study.
"""
from __future__ import annotations

import argparse
import json
import os
import statistics
import subprocess
import sys
import threading
import time

import numpy as np

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

METRIC = "grid_point_updates_per_sec"
UNIT = "GLUPS"
ESIZE = {"f32": 4, "f64": 8}


def make_cfg(name, scale=1.0):
    """BASELINE.json configs by name; `scale` < 1 shrinks the grid for the CPU samples only."""
    from paper_1310_3422_b200 import inputs
    if name == "c1":
        return inputs.make_c1()
    if name == "c2":
        return inputs.make_c2(n=int(2 ** 20 * scale))
    if name == "c3":
        return inputs.make_c3(batch=max(1, int(4096 * scale)))
    if name == "c4":
        return inputs.make_c4(n=int(2 ** 28 * scale))
    if name in ("c5_f32", "c5_f64"):
        n = int(8192 * scale ** 0.5)
        return inputs.make_c5(n=n - n % 2, dtype=name[3:])
    if name == "paper":                       # PAPER.md:204-218 run shape; use with --k 16
        return inputs.make_paper()
    if name in ("box_f32", "box_f64"):        # 3-D (NEXT-4), not a BASELINE.json config
        n = int(int(os.environ.get("GE_BOX_N", "512")) * scale ** (1.0 / 3.0))
        return inputs.make_box(n=n - n % 2, dtype=name[4:])
    raise SystemExit("unknown --config %s" % name)


def units(cfg, levels=None):
    """grid-point updates of one step"""
    lv = cfg["steps"] if levels is None else levels
    return cfg["nx"] * cfg["ny"] * cfg.get("nz", 1) * cfg["batch"] * lv


def workload_desc(cfg):
    if cfg["dim"] == 3:
        shape = "%dx%dx%d" % (cfg["nz"], cfg["ny"], cfg["nx"])
    elif cfg["dim"] == 2:
        shape = "%dx%d" % (cfg["ny"], cfg["nx"])
    elif cfg["batch"] > 1:
        shape = "%d rods x %d" % (cfg["batch"], cfg["nx"])
    else:
        shape = "N=%d" % cfg["nx"]
    return "%s: %s-D GE, %s interior, %s, %d levels per step" % (
        cfg["name"], cfg["dim"], shape, cfg["dtype"], cfg["steps"])


# ------------------------------------------------------------------ oracle legs (CPU) ------
def oracle_time(cfg):
    """Seconds the oracle, as it stands, needs for cfg (one host thread)."""
    from oracle import ge_oracle          # allowed here only: cpu_baseline / --impl reference legs
    u0 = cfg["u0"].astype(np.float64)
    t0 = time.perf_counter()
    if cfg["dim"] == 3:
        ge_oracle.run_3d(u0, cfg["r"][0], cfg["steps"])
    elif cfg["dim"] == 2:
        ge_oracle.run_2d(u0, cfg["r"][0], cfg["steps"],
                         (cfg["bc_lo"][0], cfg["bc_hi"][0], cfg["bc_lo"][1], cfg["bc_hi"][1]))
    elif cfg["batch"] == 1:
        ge_oracle.run_1d(u0.reshape(-1), cfg["r"][0], cfg["steps"], cfg["bc_lo"][0], cfg["bc_hi"][0], k=cfg.get("k", 1))
    else:
        ge_oracle.run_batched_1d(u0, cfg["r"], cfg["steps"], cfg["bc_lo"], cfg["bc_hi"])
    return time.perf_counter() - t0


def sample_desc(cfg, scale):
    return "same recipe at 1/%d of the grid (%s), all %d levels, oracle/ge_ref.c -O2" % (
        round(1 / scale), workload_desc(cfg).split(": ")[1].split(",")[1].strip(), cfg["steps"])


def oracle_time_allcores(cfg):
    """Seconds of the all-cores timing driver (oracle/ge_ref_omp.c: the same literal formulas, the groups of
    a level split across threads; pinned bit for bit to ge_ref.c by tests/test_oracle_omp.py), or None for
    workloads it does not cover (k >= 2, 3-D)."""
    from oracle import ge_oracle_omp as om
    if cfg.get("k", 1) != 1 or cfg["dim"] == 3:
        return None, 0
    om.build()
    u0 = cfg["u0"].astype(np.float64)
    t0 = time.perf_counter()
    if cfg["dim"] == 2:
        om.run_2d(u0, cfg["r"][0], cfg["steps"], (cfg["bc_lo"][0], cfg["bc_hi"][0], cfg["bc_lo"][1], cfg["bc_hi"][1]))
    elif cfg["batch"] == 1:
        om.run_1d(u0.reshape(-1), cfg["r"][0], cfg["steps"], cfg["bc_lo"][0], cfg["bc_hi"][0])
    else:
        om.run_batched_1d(u0, cfg["r"], cfg["steps"], cfg["bc_lo"], cfg["bc_hi"])
    return time.perf_counter() - t0, om.threads()


def cpu_baseline(cfg_name, scale, k=1, levels=0, reps=2):
    """The oracle as it stands on this box's host cores, on ONE bounded sample of the workload: (a) one
    thread (the parity oracle itself), (b) all cores (the OpenMP timing driver).  `value` is leg (a)."""
    from oracle import ge_oracle
    ge_oracle.build()
    scfg = make_cfg(cfg_name, scale)
    scfg["k"] = k
    if levels:
        scfg["steps"] = levels
    ts = [oracle_time(scfg) for _ in range(reps)]
    t1 = min(ts)
    out = {"value": units(scfg) / t1 / 1e9, "unit": UNIT, "cores": 1, "kind": "oracle",
           "sample": sample_desc(scfg, scale) + ", best of %d" % reps, "seconds": t1, "seconds_each": ts}
    ta, nthreads = oracle_time_allcores(scfg)
    if ta is not None:
        ta = min(ta, oracle_time_allcores(scfg)[0])
        out["all_cores"] = {"value": units(scfg) / ta / 1e9, "unit": UNIT, "cores": nthreads,
                            "host_cores": os.cpu_count(), "kind": "oracle formulas, OpenMP over the groups of a level (oracle/ge_ref_omp.c)",
                            "sample": "the same sample", "seconds": ta}
    return out


def run_reference(args):
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    from oracle import ge_oracle
    ge_oracle.build()
    scale = args.ref_scale
    cfg = make_cfg(args.config, scale)
    for _ in range(args.warmup):
        oracle_time(cfg)
    ts = [oracle_time(cfg) for _ in range(args.steps)]
    tot = sum(ts)
    value = units(cfg) * args.steps / tot / 1e9
    full = make_cfg_meta(args.config)
    line = {
        "impl": "reference", "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": args.gpus,
        "steps": args.steps, "warmup": args.warmup, "ms_per_step": 1e3 * tot / args.steps,
        "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f64",
        "data": "synthetic",
        "config": {"workload": full, "sample": sample_desc(cfg, scale)},
        "cpu_baseline": {"value": value, "unit": UNIT, "cores": 1, "kind": "oracle",
                         "sample": sample_desc(cfg, scale) + ", 1 thread, every step one run of the sample"},
        "e2e": {"value": value, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0,
    }
    print(json.dumps(line), flush=True)


def make_cfg_meta(name):
    meta = {"c1": "c1: 1-D GE, N=64 interior, f64, 1000 levels per step",
            "c2": "c2: 1-D GE, N=1048576 interior, f64, 10000 levels per step",
            "c3": "c3: 1-D GE, 4096 rods x 4096 interior, f32, 2000 levels per step",
            "c4": "c4: 1-D GE, N=268435456 interior, f64, 200 levels per step",
            "c5_f32": "c5_f32: 2-D GE, 8192x8192 interior, f32, 1000 levels per step",
            "c5_f64": "c5_f64: 2-D GE, 8192x8192 interior, f64, 1000 levels per step",
            "paper": "paper: 1-D GE, N=8206 interior, f32, 1200 levels per step",
            "box_f32": "box_f32: 3-D GE, 512x512x512 interior, f32, 100 levels per step",
            "box_f64": "box_f64: 3-D GE, 512x512x512 interior, f64, 100 levels per step"}
    return meta[name]


# ------------------------------------------------------------------ clocks ------
class ClockSampler:
    """nvidia-smi clocks/throttle reasons during the timed region (B200_PROFILING.md clocks line)."""
    Q = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,"
         "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,"
         "clocks_event_reasons.sw_power_cap")

    def __init__(self, index):
        self.rows, self.proc, self.t0, self.t1 = [], None, None, None
        try:
            self.proc = subprocess.Popen(
                ["nvidia-smi", "-i", str(index), "--query-gpu=" + self.Q, "--format=csv,noheader,nounits",
                 "-lms", "20"], stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
            self.th = threading.Thread(target=self._pump, daemon=True)
            self.th.start()
        except OSError:
            self.proc = None

    def _pump(self):
        for ln in self.proc.stdout:
            self.rows.append((time.monotonic(), ln.strip()))

    def wait_ready(self, timeout=2.0):
        """nvidia-smi needs a few hundred ms to deliver its first row; short timed regions would see none"""
        t = time.monotonic()
        while self.proc and not self.rows and time.monotonic() - t < timeout:
            time.sleep(0.02)

    def begin(self):
        self.t0 = time.monotonic()

    def end(self):
        self.t1 = time.monotonic()

    def close(self):
        if self.proc:
            time.sleep(0.15)
            self.proc.terminate()
            try:
                self.proc.wait(timeout=5)
            except subprocess.TimeoutExpired:
                self.proc.kill()

    def summary(self):
        sm, mx, reasons = [], [], set()
        names = ("hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap")
        for t, ln in self.rows:
            if self.t0 is None or not (self.t0 <= t <= (self.t1 or t) + 0.05):
                continue
            f = [x.strip() for x in ln.split(",")]
            if len(f) < 7:
                continue
            try:
                sm.append(float(f[0])); mx.append(float(f[1]))
            except ValueError:
                continue
            for nm, v in zip(names, f[3:7]):
                if v.lower().startswith("active"):
                    reasons.add(nm)
        if not sm:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": [], "samples": 0}
        return {"sm_mhz": statistics.median(sm), "sm_max_mhz": max(mx), "reasons": sorted(reasons),
                "samples": len(sm)}


# ------------------------------------------------------------------ multi-rank plumbing ------
def max_over_ranks(ms, world, device):
    """Device time of the slowest rank (the job is as slow as its slowest replica)."""
    if world <= 1:
        return float(ms)
    import torch
    import torch.distributed as dist
    t = torch.tensor([float(ms)], dtype=torch.float64, device=device)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())


def job_value(units_per_rank_step, steps, world, ms):
    """Whole-job GLUPS: "replicas only" -- every rank marches its own copy of the workload (weak scaling),
    no data-path collective; value = updates of all ranks / max-over-ranks time."""
    return units_per_rank_step * steps * world / (ms * 1e-3) / 1e9


# ------------------------------------------------------------------ our arm (CUDA) ------
SYNC_IDS = {"flags": 0, "grid": 1, "lines": 2, "stagger": 3}


def fma_peaks(dev, stream_obj):
    """Sustained FFMA / DFMA throughput of this GPU, measured now with libge's probe kernel (8 independent
    FMA chains per thread, 2048 threads per SM): the peak the "alu"-bound rooflines are divided by
    (the lane counts are an assumption until measured)."""
    import torch
    from paper_1310_3422_b200 import libge
    sink = torch.zeros(16, dtype=torch.float64, device=dev)
    out = {}
    for dt, iters in (("f32", 1 << 17), ("f64", 1 << 16)):
        libge.ge_fma_probe(dt, 1 << 12, sink.data_ptr(), stream_obj.cuda_stream)       # warm-up
        best = 0.0
        for _ in range(3):
            e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            e0.record(stream_obj)
            flops = libge.ge_fma_probe(dt, iters, sink.data_ptr(), stream_obj.cuda_stream)
            e1.record(stream_obj)
            torch.cuda.synchronize(dev)
            best = max(best, flops / (e0.elapsed_time(e1) * 1e-3) / 1e12)
        out[dt + "_tflops"] = best
        # the same with three distinct registers per FMA (what real kernels look like to the register file): context,
        # not the roofline denominator
        libge.ge_fma_probe(dt, 1 << 12, sink.data_ptr(), stream_obj.cuda_stream, 1)
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        e0.record(stream_obj)
        flops = libge.ge_fma_probe(dt, iters, sink.data_ptr(), stream_obj.cuda_stream, 1)
        e1.record(stream_obj)
        torch.cuda.synchronize(dev)
        out[dt + "_tflops_distinct_operands"] = flops / (e0.elapsed_time(e1) * 1e-3) / 1e12
    clk = float(measured_peaks()[0].get("sm_max_mhz", 1965.0)) * 1e6
    out["derived"] = {dt + "_tflops": 2.0 * LANES[dt] * SMS * clk / 1e12 for dt in ("f32", "f64")}
    out["how"] = ("ge_fma_probe (csrc/ge_probe.cuh): 8 independent dependent-FMA chains per thread, 2048 threads per SM, "
                  "best of 3 launches of ~10 ms, CUDA events; derived = 2 flop x lanes/SM (128 f32, 64 f64) x %d SMs x %.0f MHz" % (SMS, clk / 1e6))
    return out


def pcie_rates(dev, stream_obj, nbytes=1 << 29):
    """Host<->device copy rates of this box (pinned memory, one direction at a time): the ceiling of `e2e`."""
    import torch
    h = torch.empty(nbytes, dtype=torch.uint8).pin_memory()
    d = torch.empty(nbytes, dtype=torch.uint8, device=dev)
    out = {}
    for name, fn in (("h2d_gbs", lambda: d.copy_(h, non_blocking=True)), ("d2h_gbs", lambda: h.copy_(d, non_blocking=True))):
        fn()
        torch.cuda.synchronize(dev)
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        e0.record(stream_obj)
        fn()
        e1.record(stream_obj)
        torch.cuda.synchronize(dev)
        out[name] = nbytes / (e0.elapsed_time(e1) * 1e-3) / 1e9
    # both directions at once on two streams (what a pipelined step does): the time until BOTH copies are done
    h2 = torch.empty(nbytes, dtype=torch.uint8).pin_memory()
    d2 = torch.empty(nbytes, dtype=torch.uint8, device=dev)
    s_up, s_down = torch.cuda.Stream(dev), torch.cuda.Stream(dev)
    best = None
    for _ in range(2):
        torch.cuda.synchronize(dev)
        e0, e1, e2 = (torch.cuda.Event(enable_timing=True) for _ in range(3))
        e0.record(stream_obj)
        s_up.wait_event(e0); s_down.wait_event(e0)
        with torch.cuda.stream(s_up):
            d.copy_(h, non_blocking=True); e1.record(s_up)
        with torch.cuda.stream(s_down):
            h2.copy_(d2, non_blocking=True); e2.record(s_down)
        torch.cuda.synchronize(dev)
        t = max(e0.elapsed_time(e1), e0.elapsed_time(e2))
        best = t if best is None else min(best, t)
    out["duplex_gbs_each"] = nbytes / (best * 1e-3) / 1e9
    return out


def _window_1d(oracle, u0, r, steps, lo, hi, start, width):
    """Oracle values of elements [start, start+width) after `steps` levels from level 0, marched on the
    dependency cone only (a two-point group reads u_{i-1}..u_{i+2}: at most 2 nodes per side
    and level); the sub-rod starts at an even element so that its pair pattern is the global one, a cut end
    gets an arbitrary boundary value whose influence cannot reach the window."""
    n = u0.shape[0]
    halo = 2 * steps + 4
    a = max(0, start - halo)
    a -= a % 2
    b = min(n, start + width + halo)
    out = oracle.run_1d(u0[a:b].astype(np.float64), r, steps, lo if a == 0 else 0.123, hi if b == n else -0.456)
    return out[start - a:start - a + width]


def _window_2d(oracle, u0, r, steps, bc, x0, y0, w):
    ny, nx = u0.shape
    halo = 2 * steps + 4
    ax = max(0, x0 - halo); ax -= ax % 2
    ay = max(0, y0 - halo); ay -= ay % 2
    bx, by = min(nx, x0 + w + halo), min(ny, y0 + w + halo)
    sbc = (bc[0] if ax == 0 else 0.1, bc[1] if bx == nx else -0.2, bc[2] if ay == 0 else 0.3, bc[3] if by == ny else -0.4)
    out = oracle.run_2d(u0[ay:by, ax:bx].astype(np.float64), r, steps, sbc)
    return out[y0 - ay:y0 - ay + w, x0 - ax:x0 - ax + w]


def _window_3d(oracle, u0, r, steps, bc, x0, y0, z0, w):
    nz, ny, nx = u0.shape
    halo = 2 * steps + 4
    lo = [max(0, v - halo) for v in (x0, y0, z0)]
    lo = [v - v % 2 for v in lo]
    hi = [min(n, v + w + halo) for n, v in zip((nx, ny, nz), (x0, y0, z0))]
    fake = (0.1, -0.2, 0.3, -0.4, 0.5, -0.6)          # a cut face of the sub-box: any value, the cone keeps it out
    sbc = []
    for a, n in enumerate((nx, ny, nz)):
        sbc += [bc[2 * a] if lo[a] == 0 else fake[2 * a], bc[2 * a + 1] if hi[a] == n else fake[2 * a + 1]]
    out = oracle.run_3d(u0[lo[2]:hi[2], lo[1]:hi[1], lo[0]:hi[0]].astype(np.float64), r, steps, tuple(sbc))
    return out[z0 - lo[2]:z0 - lo[2] + w, y0 - lo[1]:y0 - lo[1] + w, x0 - lo[0]:x0 - lo[0] + w]


def parity_check(cfg, plan, dev, stream, k=1, budget=4e8):
    """A run from the config's initial state in the timed launch configuration, compared with the oracle on
    sampled dependency cones (rods: whole sampled rods).  Where the cones of the full level count would cost
    more than `budget` oracle updates each (C5: 1000 levels -> 4000^2 nodes per window) the run is repeated
    with fewer levels -- the full-length comparison is tests/test_gpu_longrun.py's."""
    import torch
    from oracle import ge_oracle
    if k != 1:
        return None
    ge_oracle.build()
    tol = 1e-12 if cfg["dtype"] == "f64" else 1e-5
    levels = cfg["steps"]
    if cfg["dim"] == 3:
        while (16 + 4 * levels + 8) ** 3 * levels > budget / 20 and levels > 4:    # the 3-D oracle eliminates every group
            levels //= 2
    elif cfg["dim"] == 2:
        while (24 + 4 * levels + 8) ** 2 * levels > budget and levels > 8:
            levels //= 2
    elif cfg["dim"] == 1 and cfg["batch"] == 1:
        while (64 + 4 * levels + 8) * levels > budget and levels > 8:
            levels //= 2
    u = torch.from_numpy(cfg["u0"].reshape(-1)).to(dev)
    plan.level = 0
    plan.run(u.data_ptr(), levels, stream)
    torch.cuda.synchronize(dev)
    got = u.cpu().numpy().astype(np.float64).reshape(cfg["u0"].shape)
    del u
    rng = np.random.default_rng(12345)
    worst, what = 0.0, ""
    if cfg["dim"] == 3:
        nz, ny, nx = cfg["u0"].shape
        w = 16
        bc = (cfg["bc_lo"][0], cfg["bc_hi"][0], cfg["bc_lo"][1], cfg["bc_hi"][1], cfg["bc_lo"][2], cfg["bc_hi"][2])
        pts = [(0, 0, 0), (nx - w, ny - w, nz - w), (nx - w, 0, (nz - w) // 2)]
        pts += [tuple(int(v) for v in rng.integers(0, min(nx, ny, nz) - w, size=3)) for _ in range(2)]
        for x0, y0, z0 in pts:
            x0 -= x0 % 2; y0 -= y0 % 2; z0 -= z0 % 2
            ref = _window_3d(ge_oracle, cfg["u0"], cfg["r"][0], levels, bc, x0, y0, z0, w)
            worst = max(worst, float(np.abs(got[z0:z0 + w, y0:y0 + w, x0:x0 + w] - ref).max()))
        scale = float(np.abs(cfg["u0"]).max())
        what = "%d windows of %dx%dx%d nodes on their dependency cones" % (len(pts), w, w, w)
    elif cfg["dim"] == 2:
        ny, nx = cfg["u0"].shape
        w = 24
        bc = (cfg["bc_lo"][0], cfg["bc_hi"][0], cfg["bc_lo"][1], cfg["bc_hi"][1])
        pts = [(0, 0), (nx - w, ny - w)] + [tuple(int(v) for v in rng.integers(0, min(nx, ny) - w, size=2)) for _ in range(2)]
        for x0, y0 in pts:
            x0 -= x0 % 2; y0 -= y0 % 2
            ref = _window_2d(ge_oracle, cfg["u0"], cfg["r"][0], levels, bc, x0, y0, w)
            worst = max(worst, float(np.abs(got[y0:y0 + w, x0:x0 + w] - ref).max()))
        scale = float(np.abs(cfg["u0"]).max())
        what = "%d windows of %dx%d nodes on their dependency cones" % (len(pts), w, w)
    elif cfg["batch"] == 1:
        n, w = cfg["nx"], 64
        u0 = cfg["u0"].reshape(-1)
        g = got.reshape(-1)
        starts = [0, n - w] + [int(v) for v in rng.integers(0, n - w, size=2)] if n > 4 * w else [0]
        for st in starts:
            st -= st % 2
            ww = min(w, n - st)
            ref = _window_1d(ge_oracle, u0, cfg["r"][0], levels, cfg["bc_lo"][0], cfg["bc_hi"][0], st, ww)
            worst = max(worst, float(np.abs(g[st:st + ww] - ref).max()))
        scale = float(np.abs(u0).max())
        what = "%d windows of %d nodes on their dependency cones" % (len(starts), w)
    else:
        rows = np.unique(np.concatenate([[0, cfg["batch"] - 1], rng.integers(0, cfg["batch"], size=2)]))
        ref = ge_oracle.run_batched_1d(cfg["u0"][rows].astype(np.float64), cfg["r"][rows], levels,
                                       cfg["bc_lo"][rows], cfg["bc_hi"][rows])
        worst = float((np.abs(got[rows] - ref).max(axis=1) / np.abs(ref).max(axis=1)).max())
        scale = 1.0
        what = "%d whole rods" % len(rows)
    err = worst / scale
    return {"rel_err": err, "tolerance": tol, "ok": bool(err <= tol), "levels": levels, "sample": what,
            "norm": "max|gpu - oracle| / max|u| (DESIGN.md reading R-A7)", "oracle": "oracle/ge_ref.c"}


def device_timing(cfg, args_like, dev, stream_obj, steps, warmup, world=1, clocks_index=None, flush_l2=False,
                  with_parity=True, k=1):
    """W warm-up steps, then K timed steps of ge_run on a device-resident state; returns the measurement dict
    and the plan (open) for the caller's further legs."""
    import torch
    import torch.distributed as dist
    from paper_1310_3422_b200 import libge
    stream = stream_obj.cuda_stream
    levels = cfg["steps"]

    def barrier():
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize(dev)

    u = torch.from_numpy(cfg["u0"].reshape(-1)).to(dev)
    plan = libge.Plan(cfg, kernel=args_like.get("kernel", "auto"), tb=args_like.get("tb", 0), stream=stream, group_k=k)
    for key, what in (("tc", libge.GE_TUNE_TEMPORAL_C), ("rc", libge.GE_TUNE_RESIDENT_C), ("hl", libge.GE_TUNE_HALO_LANES)):
        if args_like.get(key):
            plan.tune(what, args_like[key])
    if args_like.get("hp"):
        plan.tune(libge.GE_TUNE_SEG_PAIRS, args_like["hp"])
    if args_like.get("coop") is not None and args_like.get("coop") >= 0:
        plan.tune(libge.GE_TUNE_STRIP_COOP, args_like["coop"])
    if args_like.get("kform") is not None and args_like.get("kform") >= 0 and k >= 2:
        plan.tune(libge.GE_TUNE_K_FORM, args_like["kform"])
    if args_like.get("form3d") is not None and args_like.get("form3d") >= 0:
        plan.tune(libge.GE_TUNE_FORM_3D, args_like["form3d"])
    if args_like.get("sync"):
        plan.tune(libge.GE_TUNE_SYNC_MODE, SYNC_IDS[args_like["sync"]])
    if args_like.get("rtb"):
        plan.tune(libge.GE_TUNE_TB, args_like["rtb"])
    info0 = plan.info()
    flush = torch.empty(1 << 28, dtype=torch.uint8, device=dev) if flush_l2 else None     # 256 MiB > 126 MB of L2
    clocks = ClockSampler(clocks_index) if clocks_index is not None else None     # started early: nvidia-smi needs ~0.2 s
    for _ in range(warmup):
        plan.run(u.data_ptr(), levels, stream)
    barrier()
    l0, m0 = plan.info()["launches"], plan.info()["meetings"]
    e0 = [torch.cuda.Event(enable_timing=True) for _ in range(steps)]
    e1 = [torch.cuda.Event(enable_timing=True) for _ in range(steps)]
    barrier()
    if clocks:
        clocks.wait_ready()
        clocks.begin()
    for i in range(steps):
        if flush is not None:
            flush.zero_()
        e0[i].record(stream_obj)
        plan.run(u.data_ptr(), levels, stream)
        e1[i].record(stream_obj)
    barrier()
    if clocks:
        clocks.end()
    per_step = [e0[i].elapsed_time(e1[i]) for i in range(steps)]
    # consecutive steps without a flush: the whole bracket (first start to last end); with a flush between
    # the steps: the sum of the steps' own intervals (the flush is not part of the workload)
    total_ms = sum(per_step) if flush is not None else e0[0].elapsed_time(e1[-1])
    launches = plan.info()["launches"] - l0
    meetings = plan.info()["meetings"] - m0
    total_ms_max = max_over_ranks(total_ms, world, dev)
    finite = bool(torch.isfinite(u).all().item())
    fault = plan.sync_fault() if info0["resident_path"] == 2 else 0
    del u, flush
    if clocks:
        clocks.close()
    info0["group_k"] = k
    info0["form3d"] = 0 if args_like.get("form3d") == 0 else 1
    info0["kform"] = 0 if args_like.get("kform") == 0 else 1
    out = {"value": job_value(units(cfg), steps, world, total_ms_max), "ms_per_step": total_ms_max / steps,
           "total_ms_this_rank": total_ms, "per_step": per_step, "launches": launches, "meetings": meetings,
           "finite": finite and not fault, "info": info0, "clocks": clocks.summary() if clocks else None,
           "l2": "flushed between timed steps (256 MiB write)" if flush_l2 else None}
    return out, plan


def run_ours(args):
    import torch
    import torch.distributed as dist
    from paper_1310_3422_b200 import build as gebuild, libge

    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device; the product path has no CPU fallback")
    if rank == 0:
        gebuild.build()
    torch.cuda.set_device(local)
    dev = torch.device("cuda", local)
    if world > 1:
        dist.init_process_group("nccl", device_id=dev)
        dist.barrier()
    libge.load()
    stream_obj = torch.cuda.current_stream(dev)
    stream = stream_obj.cuda_stream

    def barrier():
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize(dev)

    peaks_alu = fma_peaks(dev, stream_obj)
    tune = dict(kernel=args.kernel, tb=args.tb, tc=args.tc, rc=args.rc, hl=args.hl, sync=args.sync, rtb=args.rtb,
                hp=args.hp, coop=args.coop, form3d=args.form3d, kform=args.kform)

    cfg = make_cfg(args.config)
    if args.levels:
        cfg["steps"] = args.levels
    levels = cfg["steps"]
    es = ESIZE[cfg["dtype"]]
    nelem = cfg["nx"] * cfg["ny"] * cfg.get("nz", 1) * cfg["batch"]
    fits_l2 = nelem * es <= 126e6

    # ---- device-resident timing: W warm-up steps, then exactly K timed steps ----
    m, plan = device_timing(cfg, tune, dev, stream_obj, args.steps, args.warmup, world=world,
                            clocks_index=local if rank == 0 else None, flush_l2=fits_l2, k=args.k)
    info0 = m["info"]
    roof = roofline(cfg, info0, m["total_ms_this_rank"], m["launches"], args.steps, peaks_alu)

    # ---- end to end through the C ABI with HOST buffers (pinned), copies inside the timed region ----
    e2e = None
    if not args.no_e2e:
        hbuf = torch.from_numpy(cfg["u0"].reshape(-1)).clone().pin_memory()
        plan.level = 0
        for _ in range(args.warmup):
            plan.run_host(hbuf.data_ptr(), levels, stream)
        barrier()
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        t0 = time.perf_counter()
        e0.record(stream_obj)
        for _ in range(args.steps):
            plan.run_host(hbuf.data_ptr(), levels, stream)     # H2D + levels + D2H + stream sync
        e1.record(stream_obj)
        barrier()
        ms = e0.elapsed_time(e1)
        wall = (time.perf_counter() - t0) * 1e3
        tt = max_over_ranks(max(ms, wall), world, dev)
        e2e = {"value": job_value(units(cfg), args.steps, world, tt), "unit": UNIT,
               "h2d_bytes_per_step": nelem * es, "d2h_bytes_per_step": nelem * es,
               "steps": args.steps, "warmup": args.warmup, "ms_per_step": tt / args.steps}
        del hbuf
        if rank == 0:
            pc = pcie_rates(dev, stream_obj)
            # uploads and downloads overlap (ge_run_host pipelines chunks): the slower direction is the floor
            floor_ms = max(nelem * es / pc["h2d_gbs"], nelem * es / pc["d2h_gbs"]) / 1e6
            duplex_ms = nelem * es / pc["duplex_gbs_each"] / 1e6
            e2e["pcie"] = dict(pc, ceiling_ms_per_step=floor_ms, frac_of_ceiling=floor_ms / (tt / args.steps),
                               duplex_ceiling_ms_per_step=duplex_ms, frac_of_duplex_ceiling=duplex_ms / (tt / args.steps),
                               note="measured on this box with pinned 512 MiB copies: one direction at a time (the step "
                                    "cannot be faster than its slower copy direction), and both directions at once on two "
                                    "streams (duplex_gbs_each: the rate each direction gets then, which is what a "
                                    "pipelined step can reach)")

    # ---- oracle legs on this box's host cores (rank 0, N = 1 only): parity of the timed configuration, CPU baseline ----
    parity, cpu = None, None
    if rank == 0 and world == 1 and not args.no_cpu:
        parity = parity_check(cfg, plan, dev, stream, k=args.k)
        cpu = cpu_baseline(args.config, args.cpu_scale, k=args.k, levels=args.levels)
    info = plan.info()
    plan.close()

    # ---- the other single-GPU configs, device-resident (rank 0, N = 1, default workload only) ----
    secondary = None
    if rank == 0 and world == 1 and args.config == "c4" and not args.no_secondary and args.kernel == "auto" and not args.levels:
        secondary = {}
        for name in ("c5_f32", "c5_f64", "c2", "c3", "box_f32", "box_f64"):
            scfg = make_cfg(name)
            sn = scfg["nx"] * scfg["ny"] * scfg.get("nz", 1) * scfg["batch"] * ESIZE[scfg["dtype"]]
            sm_, splan = device_timing(scfg, {}, dev, stream_obj, 3, 3, clocks_index=local, flush_l2=sn <= 126e6)
            sroof = roofline(scfg, sm_["info"], sm_["total_ms_this_rank"], sm_["launches"], 3, peaks_alu)
            spar = parity_check(scfg, splan, dev, stream) if not args.no_cpu else None
            splan.close()
            secondary[name] = {"workload": workload_desc(scfg), "value": sm_["value"], "unit": UNIT, "steps": 3, "warmup": 3,
                               "ms_per_step": sm_["ms_per_step"], "ms_per_step_each": sm_["per_step"],
                               "kernel": sroof["kernel"], "gpu_launches": sm_["launches"], "finite": sm_["finite"],
                               "effective_gbs": sm_["value"] * 2 * ESIZE[scfg["dtype"]], "l2": sm_["l2"],
                               "roofline": {kk: sroof.get(kk) for kk in ("bound", "achieved", "peak", "unit", "frac", "issue_frac", "peak_source", "ms_per_launch", "levels_per_launch")},
                               "parity": spar, "clocks": sm_["clocks"]}
            del scfg

    if rank != 0:
        if world > 1:
            dist.destroy_process_group()
        return

    line = {
        "metric": METRIC, "value": m["value"], "unit": UNIT, "n_gpus": world, "steps": args.steps,
        "warmup": args.warmup, "ms_per_step": m["ms_per_step"], "higher_is_better": True,
        "scaling": "weak", "vs_baseline": None, "dtype": cfg["dtype"], "data": "synthetic",
        "config": {"workload": workload_desc(cfg), "levels_per_step": levels, "kernel": info["kernel"],
                   "group_k": args.k, "tb": info["resident_tb"] if info["resident_path"] == 2 else (0 if info["resident_path"] else info["tb"]),
                   "resident": {"path": info["resident_path"], "c": info["resident_c"],
                                "warps": info["resident_warps"], "capacity": info["resident_capacity"],
                                "meetings_per_step": m["meetings"] // max(1, args.steps),
                                "sync": args.sync or "grid"} if info["resident_path"] else None,
                   "parallelism": "replicas only" if world > 1 else "single GPU",
                   "l2": "state %.0f MiB %s L2 (126 MB)%s" % (nelem * es / 2 ** 20, "fits in" if fits_l2 else "larger than",
                                                             "; " + m["l2"] if m["l2"] else "; no flush needed"),
                   "state": "consecutive: step i starts from the end state of step i-1 (the cost of a level does not depend on the data); parity is checked on a separate run from u0",
                   "r": float(cfg["r"][0]) if cfg["batch"] == 1 else "per rod U[0.5,8]"},
        "effective_gbs": m["value"] * 2 * es,            # what one-round-trip-per-level would have had to move
        "ms_per_step_each": m["per_step"],
        "finite": m["finite"],
        "parity": parity,
        "gpu_launches": m["launches"],
        "roofline": roof,
        "alu_peaks": peaks_alu,
        "e2e": e2e,
        "cpu_baseline": cpu,
        "clocks": m["clocks"],
        "secondary": secondary,
    }
    print(json.dumps(line), flush=True)
    if world > 1:
        dist.destroy_process_group()


def run_sweep(args):
    """Synchronisation study on B200: the paper asks where the barriers of its threaded
    loop must go (Fig 3) and sweeps the number of virtual blocks (Fig 4).
    The analogue here, on one long rod that fits on the chip (BASELINE.json configs[1], C2): launch per level
    (strategy A) / per tb levels (B) / one cooperative launch (C) with its kinds of meeting; tile size (values
    per lane C), halo lanes and meeting interval of strategy C.  One line per setting; every setting runs the
    same seeded input and must reproduce the first one bit for bit.  `--md FILE` also writes a markdown table."""
    import torch
    from paper_1310_3422_b200 import build as gebuild, inputs, libge
    gebuild.build()
    libge.load()
    dev = torch.device("cuda:0")
    n, levels, reps = args.sweep_n, args.levels or 10000, max(3, args.steps if args.steps != 20 else 5)
    cfg = inputs.make_c2(n=n, steps=levels)
    stream_obj = torch.cuda.current_stream(dev)
    stream = stream_obj.cuda_stream
    u0 = torch.from_numpy(cfg["u0"].reshape(-1)).to(dev)
    sync_names = {libge.GE_SYNC_FLAGS: "flag + fence", libge.GE_SYNC_GRID: "grid barrier",
                  libge.GE_SYNC_LINES: "flag-in-data", libge.GE_SYNC_STAGGER: "staggered flag-in-data",
                  libge.GE_SYNC_CLUSTER2: "clusters of 2 (DSMEM)", libge.GE_SYNC_CLUSTER4: "clusters of 4 (DSMEM)",
                  libge.GE_SYNC_CLUSTER8: "clusters of 8 (DSMEM)", libge.GE_SYNC_CLUSTER16: "clusters of 16 (DSMEM)"}
    settings = [("A: launch per level", dict(kernel="per_step"), {}),
                ("B: warp-per-tile, tb 16", dict(kernel="temporal", tb=16), {libge.GE_TUNE_TEMPORAL_C: 16}),
                ("B: TMA-staged, tb 20", dict(kernel="temporal", tb=20), {})]
    for c in (16, 32, 64):
        for hl in (1, 2, 3):
            for sync in (libge.GE_SYNC_FLAGS, libge.GE_SYNC_GRID, libge.GE_SYNC_LINES):
                settings.append(("C: C=%d, halo %d, %s" % (c, hl, sync_names[sync]), dict(kernel="persistent"),
                                 {libge.GE_TUNE_RESIDENT_C: c, libge.GE_TUNE_HALO_LANES: hl,
                                  libge.GE_TUNE_SYNC_MODE: sync}))
    for tb in (8, 16, 32):
        for sync in (libge.GE_SYNC_FLAGS, libge.GE_SYNC_GRID, libge.GE_SYNC_LINES):
            settings.append(("C: C=32, halo 2, %s, tb %d" % (sync_names[sync], tb), dict(kernel="persistent"),
                             {libge.GE_TUNE_RESIDENT_C: 32, libge.GE_TUNE_HALO_LANES: 2,
                              libge.GE_TUNE_SYNC_MODE: sync, libge.GE_TUNE_TB: tb}))
    for c, hl in ((32, 2), (32, 1), (64, 2)):
        settings.append(("C: C=%d, halo %d, %s" % (c, hl, sync_names[libge.GE_SYNC_STAGGER]), dict(kernel="persistent"),
                         {libge.GE_TUNE_RESIDENT_C: c, libge.GE_TUNE_HALO_LANES: hl,
                          libge.GE_TUNE_SYNC_MODE: libge.GE_SYNC_STAGGER}))
    # thread-block clusters: shared memory + the cluster barrier inside a cluster, flags between clusters
    for c, hl in ((32, 2), (32, 1), (16, 2), (64, 2)):
        for sync in (libge.GE_SYNC_CLUSTER2, libge.GE_SYNC_CLUSTER4, libge.GE_SYNC_CLUSTER8, libge.GE_SYNC_CLUSTER16):
            settings.append(("C: C=%d, halo %d, %s" % (c, hl, sync_names[sync]), dict(kernel="persistent"),
                             {libge.GE_TUNE_RESIDENT_C: c, libge.GE_TUNE_HALO_LANES: hl, libge.GE_TUNE_SYNC_MODE: sync}))
    for tb in (8, 16, 32):
        for sync in (libge.GE_SYNC_CLUSTER4, libge.GE_SYNC_CLUSTER8):
            settings.append(("C: C=32, halo 2, %s, tb %d" % (sync_names[sync], tb), dict(kernel="persistent"),
                             {libge.GE_TUNE_RESIDENT_C: 32, libge.GE_TUNE_HALO_LANES: 2,
                              libge.GE_TUNE_SYNC_MODE: sync, libge.GE_TUNE_TB: tb}))
    rows, first = [], None
    for name, kw, tune in settings:
        try:
            plan = libge.Plan(cfg, stream=stream, **kw)
            for what, value in tune.items():
                plan.tune(what, value)
        except libge.GeError as e:
            print("%-44s skipped (%s)" % (name, e))
            continue
        u = u0.clone()
        plan.run(u.data_ptr(), levels, stream)          # warm-up, and the result to compare
        torch.cuda.synchronize(dev)
        res = u.cpu().numpy()
        if first is None:
            first = res
        same = bool(np.array_equal(res, first))
        ts = []
        m0 = plan.info()["meetings"]
        for _ in range(reps):
            plan.level = 0
            u.copy_(u0)
            e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            e0.record(stream_obj)
            plan.run(u.data_ptr(), levels, stream)
            e1.record(stream_obj)
            torch.cuda.synchronize(dev)
            ts.append(e0.elapsed_time(e1))
        info = plan.info()
        meetings = (info["meetings"] - m0) // reps
        fault = plan.sync_fault() if info["resident_path"] == 2 else 0
        plan.close()
        ms = statistics.median(ts)
        glups = n * levels / ms / 1e6
        rows.append((name, info["kernel"], info["resident_tb"] or info["tb"], meetings, info["resident_warps"], ms,
                     glups, same and not fault))
        print("%-44s %-10s tb %3d meetings %5d tiles %5d  %8.3f ms  %8.1f GLUPS  %s" % (
            name, info["kernel"], rows[-1][2], meetings, info["resident_warps"], ms, glups,
            "bit-identical" if rows[-1][-1] else "MISMATCH"), flush=True)
    if args.md:
        with open(args.md, "w") as f:
            f.write("| setting | kernel | tb | meetings per run | tiles (warps) | tiles per SM | ms per run | GLUPS | bit-identical |\n|---|---|---|---|---|---|---|---|---|\n")
            for r in rows:
                f.write("| %s | %s | %d | %d | %d | %.2f | %.3f | %.1f | %s |\n" % (r[0], r[1], r[2], r[3], r[4], r[4] / float(SMS), r[5], r[6],
                                                                             "yes" if r[7] else "NO"))
    if not all(r[-1] for r in rows):
        raise SystemExit(1)


def run_src(args):
    """NEXT-3 measurement on the C4-shaped rod: the source term + moving boundary values (--src) or variable diffusivity
    (--var), temporally blocked through ge_run_src / ge_run_var (stationary data, 16 levels per launch) or, with
    --kernel per_step, one launch of ge_step_1d_src / ge_step_1d_var per level (HBM-bound: 3*sizeof(T) algorithmic bytes
    per update -- u in, tau*f or the link numbers in, u out)."""
    import torch
    from paper_1310_3422_b200 import build as gebuild, libge
    gebuild.build()
    libge.load()
    dev = torch.device("cuda", 0)
    cfg = make_cfg(args.config)
    levels = args.levels or cfg["steps"]
    es = ESIZE[cfg["dtype"]]
    stream_obj = torch.cuda.current_stream(dev)
    stream = stream_obj.cuda_stream
    u = torch.from_numpy(cfg["u0"].reshape(-1)).to(dev)
    v = torch.empty_like(u)
    n = cfg["nx"]
    per_level = args.kernel == "per_step"
    what = "var" if args.var else "src"
    if args.var:
        data = torch.full((n + 1,), 2.0, dtype=u.dtype, device=dev)
        data += 0.5 * torch.sin(torch.arange(n + 1, device=dev, dtype=u.dtype) * 1e-3)
    else:
        data = torch.full_like(u, 1e-9)
    lo = [1e-3 * i for i in range(levels + 1)]
    hi = [-1e-3 * i for i in range(levels + 1)]
    plan = libge.Plan(cfg, kernel="per_step", stream=stream)

    def step():
        if per_level:
            a, b = u, v
            for i in range(levels):
                if args.var:
                    plan.step_var(a.data_ptr(), b.data_ptr(), data.data_ptr(), stream)
                else:
                    plan.step_src(a.data_ptr(), b.data_ptr(), data.data_ptr(), (lo[i], lo[i + 1], hi[i], hi[i + 1]), stream)
                a, b = b, a
        elif args.var:
            plan.run_var(u.data_ptr(), levels, data.data_ptr(), stream)
        else:
            plan.run_src(u.data_ptr(), levels, data.data_ptr(), 0, lo, hi, stream)
    for _ in range(args.warmup):
        step()
    torch.cuda.synchronize(dev)
    l0 = plan.info()["launches"]
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    e0.record(stream_obj)
    for _ in range(args.steps):
        step()
    e1.record(stream_obj)
    torch.cuda.synchronize(dev)
    ms = e0.elapsed_time(e1)
    launches = plan.info()["launches"] - l0
    peaks, srcp = measured_peaks()
    upd = n * levels * args.steps
    glups = upd / (ms * 1e-3) / 1e9
    kname = ("ge1d_level_%s_kernel" % what if per_level else "ge1d_window_kernel[%s]" % what) + "<%s>" % cfg["dtype"]
    if per_level:
        gbs = 3.0 * es * glups
        roof = {"kernel": kname, "bound": "hbm", "achieved": gbs, "peak": peaks["hbm_gbs"], "unit": "GB/s", "frac": gbs / peaks["hbm_gbs"],
                "traffic": traffic_of("%s/%s" % (cfg["name"], kname)), "peak_source": srcp, "algorithmic_bytes_per_launch": 3.0 * es * n}
    elif n % (16 // es) == 0 and n >= 32 * (64 // es):
        # stationary source on rows of whole vectors: the register form (ge_temporal_src.cuh), bound by the fp pipes --
        # the factored form's 5 flops per update + the source added to each right-hand side
        lv = levels * args.steps / max(launches, 1)
        kname = "ge1d_temporal_%s_kernel<%s>" % (what, cfg["dtype"])
        alu = fma_peaks(dev, stream_obj)
        tfl = (5.0 if args.var else 6.0) * glups / 1e3
        peak = alu[cfg["dtype"] + "_tflops"]
        roof = {"kernel": kname, "bound": "alu", "achieved": tfl, "peak": peak, "unit": "TFLOP/s", "frac": tfl / peak,
                "traffic": None, "peak_source": "measured (in-run FMA microbenchmark, ge_fma_probe)", "levels_per_launch": lv,
                "algorithmic_bytes_per_launch": 3.0 * es * n, "effective_gbs": 2.0 * es * glups,
                "effective_frac_of_hbm": 2.0 * es * glups / peaks["hbm_gbs"],
                "note": "flops per update: 4 FMA + 2 ADD per pair of the factored form (5 per node), + 1 ADD per node for tau*f "
                        "(source); variable diffusivity: the same 5 with per-link coefficients from registers"}
    else:
        # blocked: HBM sees (2 u + 1 data) * sizeof(T) per node and launch of <= 16 levels; the kernel is bound by shared memory
        lv = levels * args.steps / max(launches, 1)
        gbs = 3.0 * es * glups / lv
        roof = {"kernel": kname, "bound": "hbm", "achieved": gbs, "peak": peaks["hbm_gbs"], "unit": "GB/s", "frac": gbs / peaks["hbm_gbs"],
                "traffic": None, "peak_source": srcp, "levels_per_launch": lv, "algorithmic_bytes_per_launch": 3.0 * es * n,
                "note": "shared-memory bound (two 8-byte reads and one write per node update plus the data window), not HBM-bound: "
                        "frac says how far from the HBM roof the blocked kernel runs", "effective_gbs": 2.0 * es * glups,
                "effective_frac_of_hbm": 2.0 * es * glups / peaks["hbm_gbs"]}
    print(json.dumps({
        "metric": METRIC, "value": glups, "unit": UNIT, "n_gpus": 1, "steps": args.steps,
        "warmup": args.warmup, "ms_per_step": ms / args.steps, "higher_is_better": True, "scaling": "weak",
        "vs_baseline": None, "dtype": cfg["dtype"], "data": "synthetic",
        "config": {"workload": workload_desc(cfg) + (", variable diffusivity (NEXT-3)" if args.var else ", source term + moving boundary values (NEXT-3)"),
                   "levels_per_step": levels, "kernel": "per_step" if per_level else "temporal"},
        "gpu_launches": launches, "finite": bool(torch.isfinite(u).all().item()),
        "roofline": roof, "e2e": None, "cpu_baseline": None}), flush=True)
    plan.close()


def measured_peaks():
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(p):
        with open(p) as f:
            return json.load(f), "measured (MEASURED_PEAKS.json)"
    return {"hbm_gbs": 6650.0, "sm_max_mhz": 1965.0}, "fallback (B200_PROFILING.md)"


# fp32 / fp64 lanes per SM and the SM count the ALU peak is derived from
LANES = {"f32": 128, "f64": 64}
SMS = 148
# floating-point instructions and flops (FMA = 2) per node update of the factored forms
INSTR = {1: 3.0, 2: 6.75}
FLOPS = {1: 5.0, 2: 9.75}


def traffic_of(kernel_key):
    """dram__bytes_read.sum + dram__bytes_write.sum per launch from the committed ncu --set full
    captures (profiles/traffic.json), or None when this kernel/workload has not been captured."""
    p = os.path.join(ROOT, "profiles", "traffic.json")
    if not os.path.exists(p):
        return None
    with open(p) as f:
        return json.load(f).get(kernel_key, {}).get("dram_bytes_per_launch")


def roofline(cfg, info, total_ms, launches, steps, alu=None):
    """The step is `launches/steps` launches of ONE kernel; its average duration is the CUDA-event
    time of the timed region divided by the launches in it.  Per-level kernel: HBM-bound, achieved =
    algorithmic bytes (2*sizeof(T) per update) per second against the measured copy
    rate.  Temporally blocked and resident kernels: bound by the plain fp32/fp64 pipes, achieved =
    flops of the factored form per second against 2 x lanes x SMs x max clock."""
    es = ESIZE[cfg["dtype"]]
    nelem = cfg["nx"] * cfg["ny"] * cfg.get("nz", 1) * cfg["batch"]
    peaks, src = measured_peaks()
    kernel = info["kernel"]
    ms = total_ms / max(launches, 1)
    lv = cfg["steps"] * steps / max(launches, 1)            # levels per launch (average)
    upd = nelem * lv                                        # updates per launch
    names = {"per_step": "ge%dd_level_kernel", "temporal": "ge%dd_temporal_kernel"}
    gk = info.get("group_k", 1)
    if gk >= 2:
        names["per_step"] = "ge%dd_level_k_kernel"
        names["temporal"] = "ge%dd_temporal_k_kernel" if info.get("kform") == 0 or gk not in (2, 4, 8, 16, 32) else "ge%dd_unit_k_kernel"
    if cfg["dim"] == 3:
        names["per_step"] = "ge%dd_stream_kernel+shell" if info.get("form3d", 1) else "ge%dd_level_kernel"
    if kernel == "persistent":
        name = {1: "ge1d_rod_resident_kernel", 2: "ge1d_grid_resident_kernel", 3: "ge1d_rod_k_resident_kernel"}[info["resident_path"]]
    elif kernel == "temporal" and gk == 1 and info.get("temporal_c") in (18, 22, 26, 36, 44, 52):
        name = "ge1d_stream_kernel"                      # the TMA-staged form of strategy B
    elif kernel == "temporal" and cfg["dim"] == 2 and cfg["nx"] % 4 == 0 and cfg["nx"] >= 128:
        name = "ge2d_strip_kernel"                       # the drift-free form of strategy B in 2-D
    else:
        name = names[kernel] % cfg["dim"]
    name = "%s<%s>" % (name, cfg["dtype"])
    key = "%s/%s" % (cfg["name"], name)
    eff = 2.0 * es * upd / (ms * 1e-3) / 1e9
    out = {"kernel": name, "levels_per_launch": lv, "launches_timed": launches, "ms_per_launch": ms,
           "traffic": traffic_of(key), "traffic_source": "profiles/traffic.json: dram bytes read + written per launch from a separate `ncu --set full` capture of this kernel on this workload (not measured in this run)",
           "peak_source": src,
           "algorithmic_bytes_per_launch": 2.0 * es * upd, "effective_gbs": eff,
           "effective_frac_of_hbm": eff / peaks["hbm_gbs"]}
    if kernel == "per_step" or lv <= 1.0:
        out.update({"bound": "hbm", "achieved": eff, "peak": peaks["hbm_gbs"], "unit": "GB/s",
                    "frac": eff / peaks["hbm_gbs"]})
    else:
        clk = float(peaks.get("sm_max_mhz", 1965.0)) * 1e6
        derived = 2.0 * LANES[cfg["dtype"]] * SMS * clk / 1e12
        measured = (alu or {}).get(cfg["dtype"] + "_tflops")
        peak = measured or derived
        # k >= 2: a Saul'yev node is (new - old) + (old' - old), fma: 3 instructions, 4 flops; pairs as for k = 1
        flops = FLOPS[cfg["dim"]] if gk == 1 else (4.0 * (gk - 1) + 5.0) / gk
        instr = INSTR[cfg["dim"]] if gk == 1 else (3.0 * (gk - 1) + 3.0) / gk
        ach = flops * upd / (ms * 1e-3) / 1e12
        # issue terms: FP instructions of the factored form per second against the probe's FMA instructions per second
        out.update({"bound": "alu", "achieved": ach, "peak": peak, "unit": "TFLOP/s", "frac": ach / peak,
                    "issue_frac": instr * upd / (ms * 1e-3) / (peak * 1e12 / 2.0),
                    "peak_source": "measured (in-run FMA microbenchmark, ge_fma_probe)" if measured else "derived",
                    "peak_derived": derived,
                    "peak_derivation": "2 flop x %d %s lanes/SM x %d SMs x %.0f MHz" % (
                        LANES[cfg["dtype"]], cfg["dtype"], SMS, clk / 1e6)})
    return out


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=20)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--config", default="c4")
    ap.add_argument("--kernel", default="auto")
    ap.add_argument("--tb", type=int, default=0)
    ap.add_argument("--k", type=int, default=1, help="sub-domain length (PAPER.md:82); k >= 2: per-level kernel only")
    ap.add_argument("--tc", type=int, default=0, help="1-D temporal kernel: values per lane")
    ap.add_argument("--rc", type=int, default=0, help="persistent kernels: values per lane")
    ap.add_argument("--hl", type=int, default=0, help="whole-chip persistent kernel: halo lanes per side")
    ap.add_argument("--rtb", type=int, default=0, help="whole-chip persistent kernel: levels between meetings")
    ap.add_argument("--sync", default="", choices=["", "flags", "grid", "lines", "stagger"], help="whole-chip persistent kernel: meeting kind")
    ap.add_argument("--hp", type=int, default=0, help="2-D strip kernel: output row pairs per segment")
    ap.add_argument("--coop", type=int, default=-1, help="2-D strip kernel: warps sharing one strip (0, 4, 8; -1 = plan default)")
    ap.add_argument("--kform", type=int, default=-1, help="k >= 2 blocked kernel: 1 register-resident units, 0 shared-memory windows (-1 = plan default)")
    ap.add_argument("--form3d", type=int, default=-1, help="3-D: 1 streaming + shell kernels, 0 a thread per group (-1 = plan default)")
    ap.add_argument("--levels", type=int, default=0, help="override levels per step (experiments only)")
    ap.add_argument("--src", action="store_true", help="measure ge_run_src (source term + moving boundaries, NEXT-3; --kernel per_step: ge_step_1d_src)")
    ap.add_argument("--var", action="store_true", help="measure ge_run_var (variable diffusivity, NEXT-3; --kernel per_step: ge_step_1d_var)")
    ap.add_argument("--sweep", default="", choices=["", "sync"], help="sync: the synchronisation study on the C2-shaped rod (NEXT-2)")
    ap.add_argument("--sweep-n", type=int, default=2 ** 20, help="--sweep: nodes of the rod")
    ap.add_argument("--md", default="", help="--sweep: also write a markdown table to this file")
    ap.add_argument("--no-e2e", action="store_true")
    ap.add_argument("--no-cpu", action="store_true", help="skip the oracle legs (parity, cpu_baseline)")
    ap.add_argument("--no-secondary", action="store_true", help="skip the C5 / C2 / C3 / 3-D block of the default line")
    ap.add_argument("--cpu-scale", type=float, default=1 / 128, help="grid fraction of the cpu_baseline sample")
    ap.add_argument("--ref-scale", type=float, default=1 / 128, help="grid fraction of the --impl reference sample (the same sample)")
    args = ap.parse_args()
    if args.warmup < 3 and args.impl == "ours":
        sys.stderr.write("bench.py: warning: fewer than 3 warm-up steps; the number is not reportable\n")
    if args.sweep:
        run_sweep(args)
    elif args.src or args.var:
        run_src(args)
    elif args.impl == "reference":
        run_reference(args)
    else:
        run_ours(args)


if __name__ == "__main__":
    main()
