"""Helpers for the GPU parity tests: run libge through its C ABI on torch-owned buffers."""
import numpy as np

_TORCH_DT = {"f32": "float32", "f64": "float64"}


def run_gpu(cfg, steps, kernel="auto", tb=0, level0=0, via="run", tc=0, hp=0, rc=0, hl=0, sync=None, rtb=0,
            chunks=None, k=1, coop=None, form3d=None, kform=None):
    """Run `steps` levels on cuda:0 and return the final state as a numpy array."""
    import torch
    from paper_1310_3422_b200 import libge
    dev = torch.device("cuda:0")
    u = torch.from_numpy(np.ascontiguousarray(cfg["u0"])).to(dev)
    stream = torch.cuda.current_stream(dev).cuda_stream
    with libge.Plan(cfg, kernel=kernel, tb=tb, stream=stream, group_k=k) as plan:
        plan.level = level0
        if tc:
            plan.tune(libge.GE_TUNE_TEMPORAL_C, tc)
        if hp:
            plan.tune(libge.GE_TUNE_SEG_PAIRS, hp)
        if coop is not None:
            plan.tune(libge.GE_TUNE_STRIP_COOP, coop)
        if form3d is not None:
            plan.tune(libge.GE_TUNE_FORM_3D, form3d)
        if kform is not None:
            plan.tune(libge.GE_TUNE_K_FORM, kform)
        if rc:
            plan.tune(libge.GE_TUNE_RESIDENT_C, rc)
        if hl:
            plan.tune(libge.GE_TUNE_HALO_LANES, hl)
        if sync is not None:
            plan.tune(libge.GE_TUNE_SYNC_MODE, sync)
        if rtb:
            plan.tune(libge.GE_TUNE_TB, rtb)
        if via == "run" and chunks:
            for c in chunks:                      # the same run cut into several ge_run calls
                plan.run(u.data_ptr(), c, stream)
            assert sum(chunks) == steps
        elif via == "run":
            plan.run(u.data_ptr(), steps, stream)
        elif via == "step":
            v = torch.empty_like(u)
            for _ in range(steps):
                plan.step(u.data_ptr(), v.data_ptr(), stream)
                u, v = v, u
        elif via == "host":
            h = torch.from_numpy(np.ascontiguousarray(cfg["u0"]).copy()).pin_memory()
            plan.run_host(h.data_ptr(), steps, stream)
            assert plan.level == level0 + steps
            return h.numpy().copy(), plan.info()
        else:
            raise ValueError(via)
        torch.cuda.synchronize(dev)
        assert plan.level == level0 + steps
        info = plan.info()
        if info["resident_path"] == 2:
            assert plan.sync_fault() == 0
    return u.cpu().numpy(), info


def run_oracle(oracle, cfg, steps, level0=0, k=1):
    u0 = cfg["u0"].astype(np.float64)
    if cfg["dim"] == 3:
        bc = (cfg["bc_lo"][0], cfg["bc_hi"][0], cfg["bc_lo"][1], cfg["bc_hi"][1], cfg["bc_lo"][2], cfg["bc_hi"][2])
        return oracle.run_3d(u0, cfg["r"][0], steps, bc, level0=level0)
    if cfg["dim"] == 2:
        bc = (cfg["bc_lo"][0], cfg["bc_hi"][0], cfg["bc_lo"][1], cfg["bc_hi"][1])
        return oracle.run_2d(u0, cfg["r"][0], steps, bc, level0=level0)
    if cfg["batch"] == 1:
        return oracle.run_1d(u0.reshape(-1), cfg["r"][0], steps, cfg["bc_lo"][0], cfg["bc_hi"][0],
                             k=k, level0=level0).reshape(u0.shape)
    return oracle.run_batched_1d(u0, cfg["r"], steps, cfg["bc_lo"], cfg["bc_hi"], k=k, level0=level0)


def rel_err(got, ref):
    """max-abs error relative to max|oracle| (reading R-A7); per rod for batched input."""
    got = np.asarray(got, dtype=np.float64)
    ref = np.asarray(ref, dtype=np.float64)
    return float(np.abs(got - ref).max() / max(np.abs(ref).max(), 1e-300))


def rel_err_rows(got, ref, cfg=None):
    """Per-rod max-abs error over the scale of the rod's data: max|oracle| over the interior and, when
    cfg is given, the rod's two Dirichlet values (they are part of the solution, nodes 0 and N+1;
    without them a 1-node rod between O(1) boundary values has no meaningful scale)."""
    got = np.asarray(got, dtype=np.float64)
    ref = np.asarray(ref, dtype=np.float64)
    d = np.abs(got - ref).max(axis=1)
    s = np.maximum(np.abs(ref).max(axis=1), 1e-300)
    if cfg is not None:
        s = np.maximum(s, np.maximum(np.abs(cfg["bc_lo"]), np.abs(cfg["bc_hi"])))
    return float((d / s).max())


TOL = {"f64": 1e-12, "f32": 1e-5}     # BASELINE.json north_star


def window_1d(oracle, u0, r, steps, lo, hi, start, width, level0=0):
    """Exact oracle values of elements [start, start+width) after `steps` levels, computed on the
    dependency cone only: a two-point group reads u_{i-1}..u_{i+2}, so the cone
    widens by at most 2 nodes per side per level.  The sub-rod starts at an even element so that the
    pair pattern is the global one; a cut end gets an arbitrary constant boundary value whose
    influence cannot reach the window."""
    n = u0.shape[0]
    halo = 2 * steps + 4
    a = max(0, start - halo)
    a -= a % 2
    b = min(n, start + width + halo)
    sub = u0[a:b].astype(np.float64)
    out = oracle.run_1d(sub, r, steps, lo if a == 0 else 0.123, hi if b == n else -0.456, level0=level0)
    return out[start - a:start - a + width]


def window_2d(oracle, u0, r, steps, bc, x0, y0, w, level0=0):
    """Same on a 2-D window [y0,y0+w) x [x0,x0+w); bc = (x_lo, x_hi, y_lo, y_hi)."""
    ny, nx = u0.shape
    halo = 2 * steps + 4
    ax = max(0, x0 - halo); ax -= ax % 2
    ay = max(0, y0 - halo); ay -= ay % 2
    bx = min(nx, x0 + w + halo)
    by = min(ny, y0 + w + halo)
    sub = u0[ay:by, ax:bx].astype(np.float64)
    sbc = (bc[0] if ax == 0 else 0.1, bc[1] if bx == nx else -0.2, bc[2] if ay == 0 else 0.3, bc[3] if by == ny else -0.4)
    out = oracle.run_2d(sub, r, steps, sbc, level0=level0)
    return out[y0 - ay:y0 - ay + w, x0 - ax:x0 - ax + w]
