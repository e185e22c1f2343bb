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
        n = int(512 * scale ** (1.0 / 3.0))
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
    return "same recipe at 1/%d of the grid (%s), all %d levels, oracle/ge_ref.c -O2, 1 thread" % (
        round(1 / scale), workload_desc(cfg).split(": ")[1].split(",")[1].strip(), cfg["steps"])


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
                         "sample": sample_desc(cfg, scale)},
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

    cfg = make_cfg(args.config)
    if args.levels:
        cfg["steps"] = args.levels
    levels = cfg["steps"]
    es = ESIZE[cfg["dtype"]]
    nelem = cfg["nx"] * cfg["ny"] * cfg.get("nz", 1) * cfg["batch"]
    stream_obj = torch.cuda.current_stream(dev)
    stream = stream_obj.cuda_stream

    def barrier():
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize(dev)

    host0 = torch.from_numpy(cfg["u0"].reshape(-1))
    u = host0.to(dev)
    plan = libge.Plan(cfg, kernel=args.kernel, tb=args.tb, stream=stream, group_k=args.k)
    if args.tc:
        plan.tune(libge.GE_TUNE_TEMPORAL_C, args.tc)
    if args.rc:
        plan.tune(libge.GE_TUNE_RESIDENT_C, args.rc)
    if args.hl:
        plan.tune(libge.GE_TUNE_HALO_LANES, args.hl)
    if args.sync:
        plan.tune(libge.GE_TUNE_SYNC_MODE, {"flags": libge.GE_SYNC_FLAGS, "grid": libge.GE_SYNC_GRID, "lines": libge.GE_SYNC_LINES, "stagger": libge.GE_SYNC_STAGGER}[args.sync])
    if args.rtb:
        plan.tune(libge.GE_TUNE_TB, args.rtb)
    info0 = plan.info()

    # ---- device-resident timing: W warm-up steps, then exactly K timed steps ----
    clocks = ClockSampler(local) if rank == 0 else None       # started early: nvidia-smi needs ~0.2 s to come up
    for _ in range(args.warmup):
        plan.run(u.data_ptr(), levels, stream)
    barrier()
    l0, m0 = plan.info()["launches"], plan.info()["meetings"]
    ev = [torch.cuda.Event(enable_timing=True) for _ in range(args.steps + 1)]
    barrier()
    if clocks:
        clocks.begin()
    ev[0].record(stream_obj)
    for i in range(args.steps):
        plan.run(u.data_ptr(), levels, stream)
        ev[i + 1].record(stream_obj)
    barrier()
    if clocks:
        clocks.end()
    total_ms = ev[0].elapsed_time(ev[-1])
    per_step = [ev[i].elapsed_time(ev[i + 1]) for i in range(args.steps)]
    launches = plan.info()["launches"] - l0
    meetings = plan.info()["meetings"] - m0
    total_ms_max = max_over_ranks(total_ms, world, dev)
    value = job_value(units(cfg), args.steps, world, total_ms_max)
    finite = bool(torch.isfinite(u).all().item())

    # ---- roofline of the dominant kernel: its average launch duration over the timed region ----
    info0["group_k"] = args.k
    roof = roofline(cfg, info0, total_ms, launches, args.steps)
    fault = plan.sync_fault() if info0["resident_path"] == 2 else 0

    # ---- end to end through the C ABI with HOST buffers (pinned), copies inside the timed region ----
    e2e = None
    if not args.no_e2e:
        hbuf = host0.clone().pin_memory()
        plan.level = 0
        for _ in range(1):
            plan.run_host(hbuf.data_ptr(), levels, stream)
        barrier()
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        ksteps = max(1, min(args.steps, 3))
        t0 = time.perf_counter()
        e0.record(stream_obj)
        for _ in range(ksteps):
            plan.run_host(hbuf.data_ptr(), levels, stream)     # H2D + levels + D2H + stream sync
        e1.record(stream_obj)
        barrier()
        ms = e0.elapsed_time(e1)
        wall = (time.perf_counter() - t0) * 1e3
        tt = max_over_ranks(max(ms, wall), world, dev)
        e2e = {"value": job_value(units(cfg), ksteps, world, tt), "unit": UNIT,
               "h2d_bytes_per_step": nelem * es, "d2h_bytes_per_step": nelem * es,
               "steps": ksteps, "ms_per_step": tt / ksteps}
        del hbuf

    info = plan.info()
    plan.close()
    del u
    if clocks:
        clocks.close()

    if rank != 0:
        if world > 1:
            dist.destroy_process_group()
        return

    # ---- oracle timed beside it on this box's host cores (rank 0, N = 1 only) ----
    cpu = None
    if world == 1 and not args.no_cpu:
        from oracle import ge_oracle
        ge_oracle.build()
        scale = args.cpu_scale
        scfg = make_cfg(args.config, scale)
        scfg["k"] = args.k
        if args.levels:
            scfg["steps"] = args.levels
        t = oracle_time(scfg)
        cpu = {"value": units(scfg) / t / 1e9, "unit": UNIT, "cores": 1, "kind": "oracle",
               "sample": sample_desc(scfg, scale), "seconds": t}

    line = {
        "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps,
        "warmup": args.warmup, "ms_per_step": total_ms_max / args.steps, "higher_is_better": True,
        "scaling": "weak", "vs_baseline": None, "dtype": cfg["dtype"], "data": "synthetic",
        "config": {"workload": workload_desc(cfg), "levels_per_step": levels, "kernel": info["kernel"],
                   "group_k": args.k, "tb": info["resident_tb"] if info["resident_path"] == 2 else (0 if info["resident_path"] else info["tb"]),
                   "resident": {"path": info["resident_path"], "c": info["resident_c"],
                                "warps": info["resident_warps"], "capacity": info["resident_capacity"],
                                "meetings_per_step": meetings // max(1, args.steps),
                                "sync": args.sync or "grid"} if info["resident_path"] else None,
                   "parallelism": "replicas only" if world > 1 else "single GPU",
                   "l2": "state %.0f MiB %s L2 (126 MB)" % (nelem * es / 2 ** 20,
                                                              "larger than" if nelem * es > 126e6 else "fits in"),
                   "r": float(cfg["r"][0]) if cfg["batch"] == 1 else "per rod U[0.5,8]"},
        "effective_gbs": value * 2 * es,            # what one-round-trip-per-level would have had to move
        "ms_per_step_each": per_step,
        "finite": finite and not fault,
        "gpu_launches": launches,
        "roofline": roof,
        "e2e": e2e,
        "cpu_baseline": cpu,
        "clocks": clocks.summary() if clocks else None,
    }
    print(json.dumps(line), flush=True)
    if world > 1:
        dist.destroy_process_group()


def run_src(args):
    """NEXT-3 measurement: `levels` launches of ge_step_1d_src (source array + moving boundary values) on
    the C4-shaped rod; HBM-bound, 3*sizeof(T) algorithmic bytes per update (u in, tau*f in, u out)."""
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
    src = torch.full_like(u, 1e-9)
    plan = libge.Plan(cfg, kernel="per_step", stream=stream)

    def step():
        a, b = u, v
        for n in range(levels):
            t = 1e-3 * n
            plan.step_src(a.data_ptr(), b.data_ptr(), src.data_ptr(), (t, t + 1e-3, -t, -t - 1e-3), stream)
            a, b = b, a
    for _ in range(args.warmup):
        step()
    torch.cuda.synchronize(dev)
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    e0.record(stream_obj)
    for _ in range(args.steps):
        step()
    e1.record(stream_obj)
    torch.cuda.synchronize(dev)
    ms = e0.elapsed_time(e1)
    peaks, srcp = measured_peaks()
    upd = cfg["nx"] * levels * args.steps
    gbs = 3.0 * es * upd / (ms * 1e-3) / 1e9
    print(json.dumps({
        "metric": METRIC, "value": upd / (ms * 1e-3) / 1e9, "unit": UNIT, "n_gpus": 1, "steps": args.steps,
        "warmup": args.warmup, "ms_per_step": ms / args.steps, "higher_is_better": True, "scaling": "weak",
        "vs_baseline": None, "dtype": cfg["dtype"], "data": "synthetic",
        "config": {"workload": workload_desc(cfg) + ", source term + moving boundary values (NEXT-3)",
                   "levels_per_step": levels, "kernel": "per_step"},
        "gpu_launches": levels * args.steps, "finite": bool(torch.isfinite(u).all().item()),
        "roofline": {"kernel": "ge1d_level_src_kernel<%s>" % cfg["dtype"], "bound": "hbm", "achieved": gbs,
                     "peak": peaks["hbm_gbs"], "unit": "GB/s", "frac": gbs / peaks["hbm_gbs"],
                     "traffic": traffic_of("%s/ge1d_level_src_kernel<%s>" % (cfg["name"], cfg["dtype"])),
                     "peak_source": srcp, "algorithmic_bytes_per_launch": 3.0 * es * cfg["nx"]},
        "e2e": None, "cpu_baseline": None}), flush=True)
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


def roofline(cfg, info, total_ms, launches, steps):
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
    if info.get("group_k", 1) >= 2:
        names["per_step"] = "ge%dd_level_k_kernel"
    if kernel == "persistent":
        name = "ge1d_rod_resident_kernel" if info["resident_path"] == 1 else "ge1d_grid_resident_kernel"
    elif kernel == "temporal" and info.get("temporal_c") in (18, 22, 26, 36, 44, 52):
        name = "ge1d_stream_kernel"                      # the TMA-staged form of strategy B
    elif kernel == "temporal" and cfg["dim"] == 2 and cfg["nx"] % 4 == 0 and cfg["nx"] >= 128:
        name = "ge2d_strip_kernel"                       # the drift-free form of strategy B in 2-D
    else:
        name = names[kernel] % cfg["dim"]
    name = "%s<%s>" % (name, cfg["dtype"])
    key = "%s/%s" % (cfg["name"], name)
    eff = 2.0 * es * upd / (ms * 1e-3) / 1e9
    out = {"kernel": name, "levels_per_launch": lv, "launches_timed": launches, "ms_per_launch": ms,
           "traffic": traffic_of(key), "peak_source": src,
           "algorithmic_bytes_per_launch": 2.0 * es * upd, "effective_gbs": eff,
           "effective_frac_of_hbm": eff / peaks["hbm_gbs"]}
    if kernel == "per_step" or lv <= 1.0:
        out.update({"bound": "hbm", "achieved": eff, "peak": peaks["hbm_gbs"], "unit": "GB/s",
                    "frac": eff / peaks["hbm_gbs"]})
    else:
        clk = float(peaks.get("sm_max_mhz", 1965.0)) * 1e6
        peak = 2.0 * LANES[cfg["dtype"]] * SMS * clk / 1e12
        ach = FLOPS[cfg["dim"]] * upd / (ms * 1e-3) / 1e12
        out.update({"bound": "alu", "achieved": ach, "peak": peak, "unit": "TFLOP/s", "frac": ach / peak,
                    "issue_frac": INSTR[cfg["dim"]] * upd / (ms * 1e-3) / (LANES[cfg["dtype"]] * SMS * clk),
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
    ap.add_argument("--levels", type=int, default=0, help="override levels per step (experiments only)")
    ap.add_argument("--src", action="store_true", help="measure ge_step_1d_src (source term + moving boundaries, NEXT-3)")
    ap.add_argument("--no-e2e", action="store_true")
    ap.add_argument("--no-cpu", action="store_true")
    ap.add_argument("--cpu-scale", type=float, default=1 / 32, help="grid fraction of the cpu_baseline sample")
    ap.add_argument("--ref-scale", type=float, default=1 / 256, help="grid fraction of the --impl reference sample")
    args = ap.parse_args()
    if args.warmup < 3 and args.impl == "ours":
        sys.stderr.write("bench.py: warning: fewer than 3 warm-up steps; the number is not reportable\n")
    if args.src:
        run_src(args)
    elif args.impl == "reference":
        run_reference(args)
    else:
        run_ours(args)


if __name__ == "__main__":
    main()
