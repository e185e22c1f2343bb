"""Synchronisation study on B200: the paper asks where the barriers of its
threaded loop must go (Fig 3) and sweeps the number of virtual blocks (PAPER.md:206-214,
Fig 4).  The analogue here, on one long rod that fits on the chip (BASELINE.json configs[1], C2):

  * launch per level (strategy A) / launch per tb levels (strategy B) / one cooperative launch
    (strategy C) with the three kinds of meeting of ge_resident.cuh;
  * tile size (values per lane C), halo lanes and meeting interval of strategy C.

    python -m paper_1310_3422_b200.sweep [--n 1048576] [--levels 10000] [--reps 5] [--md out.md]

Prints one line per setting (ms per run, GLUPS, meetings) and optionally a markdown table.  Every
setting is run on the same seeded input and must reproduce the first one bit for bit."""
from __future__ import annotations

import argparse
import statistics
import sys

import numpy as np


def main():
    import torch
    from . import build, inputs, libge

    ap = argparse.ArgumentParser()
    ap.add_argument("--n", type=int, default=2 ** 20)
    ap.add_argument("--levels", type=int, default=10000)
    ap.add_argument("--reps", type=int, default=5)
    ap.add_argument("--md", default="")
    args = ap.parse_args()
    build.build()
    libge.load()
    dev = torch.device("cuda:0")
    cfg = inputs.make_c2(n=args.n, steps=args.levels)
    stream_obj = torch.cuda.current_stream(dev)
    stream = stream_obj.cuda_stream
    u0 = torch.from_numpy(cfg["u0"].reshape(-1)).to(dev)
    sync_names = {libge.GE_SYNC_FLAGS: "flag + fence", libge.GE_SYNC_GRID: "grid barrier",
                  libge.GE_SYNC_LINES: "flag-in-data", libge.GE_SYNC_STAGGER: "staggered flag-in-data"}
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
        plan.run(u.data_ptr(), args.levels, stream)          # warm-up, and the result to compare
        torch.cuda.synchronize(dev)
        res = u.cpu().numpy()
        if first is None:
            first = res
        same = bool(np.array_equal(res, first))
        ts = []
        m0 = plan.info()["meetings"]
        for _ in range(args.reps):
            plan.level = 0
            u.copy_(u0)
            e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            e0.record(stream_obj)
            plan.run(u.data_ptr(), args.levels, stream)
            e1.record(stream_obj)
            torch.cuda.synchronize(dev)
            ts.append(e0.elapsed_time(e1))
        info = plan.info()
        meetings = (info["meetings"] - m0) // args.reps
        fault = plan.sync_fault() if info["resident_path"] == 2 else 0
        plan.close()
        ms = statistics.median(ts)
        glups = args.n * args.levels / ms / 1e6
        rows.append((name, info["kernel"], info["resident_tb"] or info["tb"], meetings, info["resident_warps"], ms,
                     glups, same and not fault))
        print("%-44s %-10s tb %3d meetings %5d tiles %5d  %8.3f ms  %8.1f GLUPS  %s" % (
            name, info["kernel"], rows[-1][2], meetings, info["resident_warps"], ms, glups,
            "bit-identical" if rows[-1][-1] else "MISMATCH"), flush=True)
    if args.md:
        with open(args.md, "w") as f:
            f.write("| setting | kernel | tb | meetings per run | tiles | ms per run | GLUPS | bit-identical |\n|---|---|---|---|---|---|---|---|\n")
            for r in rows:
                f.write("| %s | %s | %d | %d | %d | %.3f | %.1f | %s |\n" % (r[0], r[1], r[2], r[3], r[4], r[5], r[6],
                                                                       "yes" if r[7] else "NO"))
    return 0 if all(r[-1] for r in rows) else 1


if __name__ == "__main__":
    sys.exit(main())
