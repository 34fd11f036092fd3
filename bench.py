#!/usr/bin/env python
"""bench.py — cell-updates/s of the fused PPM+PPB timestep on B200 (BASELINE.json metric).

  python bench.py [--gpus N] [--steps K] [--warmup W] [--workload 4|5|...] [--impl reference]

A "step" is one ppm_step = the whole hot path (three fused hydro+PPB sweeps, the CFL max-reduction folded into the
last one) over the whole synthetic grid.  value = cells * K / device time, inputs resident in HBM; the
K-step region is timed with CUDA events on the library's stream, repeated (5 times; 3 at 1024^3) and the MEDIAN
repetition is reported; every repetition is listed.  The default run times config 4 (512^3, the headline)
and then, in the same process, config 5 (1024^3) as the "also" entry — the two grids the target names.
e2e = the same metric through the C ABI with pinned HOST buffers: ppm_set_state(host) + ppm_step + ppm_get_state(host)
inside the timed region, the slabs of the upload, the step and the download pipelined on two streams.
Multi-GPU: the path is "replicas only": each rank advances its own grid, no data-path collective; value
sums the ranks' cells ("weak" scaling).

--impl reference times the fp64 CPU oracle (as it stands) on a bounded sample of the same workload.
"""
import argparse
import json
import os
import subprocess
import sys
import tempfile
import time

import numpy as np
import torch

ROOT = os.path.dirname(os.path.abspath(__file__))
sys.path.insert(0, ROOT)

from paper_1810_13416_b200 import workloads as W  # noqa: E402

METRIC = "cell-updates/s per 3-D PPM+PPB step (fp32); achieved HBM GB/s vs peak"
UNIT = "cell-updates/s"
BYTES_PER_CELL_SWEEP = 120.0      # 15 fp32 fields read + written by every sweep
BYTES_PER_CELL_SWEEP_ADVECT = 84.0   # PPB-only sweep: 1 velocity + 10 coefficients read, 10 written (the hydro fields stay in their buffer)
FLOPS_PER_CELL_SWEEP = 1307.0     # operation count of the oracle's sweep body, FMA = 2
FP32_NOMINAL_TFLOPS = 148 * 128 * 2 * 1.965e9 / 1e12   # SMs x lanes x FMA x max SM clock (B200_PROFILING.md); fallback only
# dram__bytes_read.sum + dram__bytes_write.sum per sweep launch from the committed `ncu --set full` captures, keyed by
# cells per side: (bytes, the profiles/ file it comes from).  A size with no capture reports null.
NCU_TRAFFIC = {512: (16.096e9, "profiles/r2e_final_sweeps_ncu.md (ncu --set full, 512^3)"),
               1024: (128.85e9, "profiles/r2d_sweeps_1024_ncu.md (ncu, 1024^3)")}


def _peaks():
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(p):
        try:
            return float(json.load(open(p))["hbm_gbs"]), "measured"
        except Exception:
            pass
    return 6650.0, "fallback"


def max_over_ranks(vals, ws, device=None):
    """element-wise MAX of a list of floats over all ranks (the contract's max-over-ranks timing).  Works on
    whatever backend the process group was created with (nccl on the GPU box, gloo in the CPU test)."""
    if ws <= 1:
        return [float(v) for v in vals]
    import torch.distributed as dist
    t = torch.tensor([float(v) for v in vals], dtype=torch.float64, device=device if device is not None else "cpu")
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return [float(v) for v in t.cpu()]


def aggregate_value(cells_per_rank, steps, ms, ws):
    """whole-job cell-updates/s: every rank advances its own grid (replicas only, weak scaling)"""
    return ws * cells_per_rank * steps / (ms * 1e-3)


def _dist():
    ws = int(os.environ.get("WORLD_SIZE", "1"))
    rank = int(os.environ.get("RANK", "0"))
    lr = int(os.environ.get("LOCAL_RANK", "0"))
    return ws, rank, lr


class _Clocks:
    """samples nvidia-smi clocks / throttle reasons of one GPU while the timed region runs"""
    Q = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,clocks_event_reasons.hw_thermal_slowdown,"
         "clocks_event_reasons.sw_thermal_slowdown,clocks_event_reasons.sw_power_cap")

    def __init__(self, idx):
        self.f = tempfile.NamedTemporaryFile("w+", suffix=".csv", delete=False)
        try:
            self.p = subprocess.Popen(["nvidia-smi", "-i", str(idx), "--query-gpu=" + self.Q, "--format=csv,noheader,nounits",
                                       "-lms", "20"], stdout=self.f, stderr=subprocess.DEVNULL)
        except Exception:
            self.p = None

    def stop(self):
        out = {"sm_mhz": None, "sm_max_mhz": None, "reasons": []}
        if self.p is None:
            return out
        time.sleep(0.02)
        self.p.terminate()
        try:
            self.p.wait(timeout=5)
        except Exception:
            self.p.kill()
        self.f.flush()
        self.f.seek(0)
        sm, mx, reasons = [], [], set()
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        for line in self.f.read().splitlines():
            c = [x.strip() for x in line.split(",")]
            if len(c) < 7:
                continue
            try:
                sm.append(float(c[0])); mx.append(float(c[1]))
            except ValueError:
                continue
            for nme, v in zip(names, c[3:7]):
                if v.lower().startswith("active"):
                    reasons.add(nme)
        self.f.close()
        os.unlink(self.f.name)
        if sm:
            out = {"sm_mhz": float(np.median(sm)), "sm_max_mhz": float(max(mx)), "reasons": sorted(reasons), "samples": len(sm)}
        return out


def _geometry(w):
    walls = "periodic" if all(b == 0 for b in w.bc) else ("reflecting walls" if all(b == 1 for b in w.bc) else "periodic x,y + reflecting z walls")
    grav = {None: "no gravity", 1: "plane-parallel gravity", 2: "radial gravity"}[None if not w.grav else int(w.grav["kind"])]
    return walls + " + " + grav


def _load_state(g, w, nzs):
    n = w.n
    for z0 in range(0, n, nzs):
        z1 = min(n, z0 + nzs)
        g.set_state(w.fields((0, 0, z0), (n, n, z1), device=g.device), z0=z0)


# ------------------------------------------------------------------------------------------------ oracle timings
def _time_oracle(w, side, steps, warmup):
    """the fp64 oracle as it stands, all host threads, on the whole grid of `w` (side >= w.n) or on a central window"""
    from oracle import binding as ob          # bench.py's cpu_baseline / reference legs may use oracle/
    side = min(side, w.n)
    lo = [(w.n - side) // 2] * 3
    hi = [lo[0] + side] * 3
    bc = [w.bc[k] if side == w.n else 2 for k in range(6)]
    f = w.fields(lo, hi).numpy()
    o = ob.Oracle(side, side, side, w.dx, w.gamma, bc, w.grav, org=lo, rho_floor=w.rho_floor, p_floor=w.p_floor)
    o.set_state(f)
    dt = 0.5 * o.cfl_dt(w.cfl)
    for s in range(warmup):
        o.step(dt, 0 if s % 2 == 0 else 5)
    t0 = time.perf_counter()
    for s in range(steps):
        o.step(dt, 0 if s % 2 == 0 else 5)
    t = time.perf_counter() - t0
    what = "%s %d^3 grid" % (w.name, side) if side == w.n else "central %d^3 window of %s %d^3" % (side, w.name, w.n)
    return side ** 3 * steps / t, t / steps, ob.num_threads(), "%s, %d steps after %d warm-up" % (what, steps, warmup)


def _cpu_baseline(w):
    """config 2's own grid (128^3, 10 steps) and a 256^3 grid (3 steps), one warm-up step each"""
    v1, _, cores, s1 = _time_oracle(W.make(2), 128, 10, 1)
    v2, _, _, s2 = _time_oracle(w, 256, 3, 1)
    return {"value": v1, "unit": UNIT, "cores": cores, "kind": "oracle", "sample": s1,
            "also": {"value": v2, "unit": UNIT, "sample": s2}}


def run_reference(args):
    ws, rank, _ = _dist()
    if rank != 0:
        return 0
    w = W.make(args.workload)
    val, sps, cores, sample = _time_oracle(w, args.ref_side, args.steps, args.warmup)
    line = {"impl": "reference", "metric": METRIC, "value": val, "unit": UNIT, "n_gpus": args.gpus, "steps": args.steps,
            "warmup": args.warmup, "ms_per_step": sps * 1e3, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
            "dtype": "f64", "data": "synthetic",
            "config": {"workload": "%s %d^3 (oracle on a bounded window)" % (w.name, w.n), "cfl": w.cfl},
            "cpu_baseline": {"value": val, "unit": UNIT, "cores": cores, "kind": "oracle", "sample": sample},
            "e2e": {"value": val, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
            "gpu_launches": 0}
    print(json.dumps(line))
    return 0


# ------------------------------------------------------------------------------------------------ GPU timings
def _time_steps(g, do_step, dt, K, reps, barrier):
    """`reps` repetitions of a K-step region, CUDA events on the library's stream; returns the list of ms per region"""
    out = []
    for r in range(reps):
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        barrier()
        e0.record(g.stream)
        for s in range(K):
            do_step(dt, 0 if s % 2 == 0 else 5)
        e1.record(g.stream)
        barrier()
        out.append(e0.elapsed_time(e1))
    return out


def _roofline(n, ms_per_step, advect, peak, peak_kind, fp32_peak, fp32_kind):
    ncell = n ** 3
    per_launch_s = ms_per_step * 1e-3 / 3          # the dominant kernel = the 3 sweep launches of every step
    achieved = (BYTES_PER_CELL_SWEEP_ADVECT if advect else BYTES_PER_CELL_SWEEP) * ncell / per_launch_s / 1e9
    flops_cs = 478.0 if advect else FLOPS_PER_CELL_SWEEP     # PPB-only: P2 13 + P1/P3/P4 460 + face masses 5
    alu = flops_cs * ncell / per_launch_s / 1e12
    tr = NCU_TRAFFIC.get(n) if not advect else None
    return {"bound": "hbm", "achieved": achieved, "peak": peak, "unit": "GB/s", "frac": achieved / peak,
            "traffic": tr[0] if tr else None, "traffic_from": tr[1] if tr else None, "peak_kind": "of " + peak_kind,
            "kernel": ("ppm_advect_bulk_kernel (3 launches per step; every launch moves 84 B/cell: u_d and the ten PPB coefficients in, the coefficients out)"
                       if advect else "ppm_sweep_bulk_kernel (3 launches per step; every launch moves 120 B/cell)"),
            "alu": {"achieved": alu, "peak": fp32_peak, "unit": "TFLOP/s", "frac": alu / fp32_peak, "peak_kind": fp32_kind,
                    "flops_per_cell_sweep": flops_cs}}


def _bench_grid(args, cfg, dev, lr, ws, barrier, K, reps, with_e2e):
    """times one workload on this rank's GPU; returns a dict of raw numbers (ms are per K-step region)"""
    from paper_1810_13416_b200.binding import PPM, NF, OPT_IO_PATH, OPT_FLATTEN3D
    w = W.make(cfg)
    n = w.n
    g = PPM.from_workload(w, device=dev)
    if args.chunk:
        g.set_chunk(args.chunk)
    if args.direct:
        g.set_option(OPT_IO_PATH, 1)
    if args.flatten3d:
        g.set_option(OPT_FLATTEN3D, 1)
    if args.sphere:
        g.set_sphere(0.5, (0.5, 0.5, 0.5))
    if args.two_fluid:
        g.set_two_fluid(1.4, w.gamma)        # the stable layer (FV = 1) is a gamma = 1.4 gas, the convection zone keeps 5/3
    _load_state(g, w, 8 if n >= 1024 else 32)
    dt = 0.7 * g.cfl_dt(w.cfl)       # fixed for the run: no host sync inside the timed region
    do_step = g.advect if args.advect else g.step
    Wm = max(args.warmup, 3)
    for s in range(Wm):
        do_step(dt, 0 if s % 2 == 0 else 5)
    barrier()
    clk = _Clocks(lr)
    l0 = g.launch_count()
    ms_reps = _time_steps(g, do_step, dt, K, reps, barrier)
    launches = (g.launch_count() - l0) // reps
    clocks = clk.stop()
    g.sync()                         # raises if the state flag (NaN / floor) was set
    # the same K steps with ppm_cfl_dt before each one (the configs' "dt from ppm_cfl_dt each step"): after a ppm_step
    # the maximum is already on the device (reduced inside the last sweep), so this adds one 4-byte read and a host sync
    ms_cfl = []
    for r in range(min(reps, 3)):
        e2, e3 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        barrier()
        e2.record(g.stream)
        for s in range(K):
            do_step(0.7 * g.cfl_dt(w.cfl), 0 if s % 2 == 0 else 5)
        e3.record(g.stream)
        barrier()
        ms_cfl.append(e2.elapsed_time(e3))
    # the same K steps with the uniform-FV shortcut switched off (PPM_OPT_FV_SHORTCUT = 0): every cell runs the PPB remap
    ms_noskip = []
    if not args.advect:
        from paper_1810_13416_b200.binding import OPT_FV_SHORTCUT
        g.set_option(OPT_FV_SHORTCUT, 0)
        do_step(dt, 0); do_step(dt, 5)
        ms_noskip = _time_steps(g, do_step, dt, K, min(reps, 3), barrier)
        g.set_option(OPT_FV_SHORTCUT, 1)
    fp32 = None
    try:
        fp32 = g.measure_fp32_peak()
    except Exception:
        pass
    e2e = None
    if with_e2e:
        try:
            g2 = None
            try:                                   # a second context (own buffers, own stream) for the two-context pipeline
                g2 = PPM.from_workload(w, device=dev, stream=torch.cuda.Stream(dev))
                for opt in (("set_sphere", (0.5, (0.5, 0.5, 0.5))) if args.sphere else None, ("set_two_fluid", (1.4, w.gamma)) if args.two_fluid else None):
                    if opt:
                        getattr(g2, opt[0])(*opt[1])
                if args.flatten3d:
                    g2.set_option(OPT_FLATTEN3D, 1)
            except Exception:
                g2 = None
            e2e = _time_e2e(g, do_step, dt, args.e2e_steps, barrier, n, NF, g2)
            if g2 is not None:
                g2.close()
                del g2
        except Exception as ex:                                                  # e.g. not enough pinned host memory
            e2e = {"error": str(ex)[:200]}
    g.close()
    del g
    torch.cuda.empty_cache()
    return {"w": w, "n": n, "ms_reps": ms_reps, "ms_cfl": ms_cfl, "ms_noskip": ms_noskip, "launches": launches, "clocks": clocks, "fp32": fp32,
            "e2e": e2e, "warmup": Wm}


def _time_e2e(g, do_step, dt, Ke, barrier, n, NF, g2=None):
    """host buffers through the C ABI, copies inside the timed region.
    serial   : ppm_set_state(host) -> ppm_step -> ppm_get_state(host), one grid after the other on one stream;
    pipelined: a stream of INDEPENDENT host-resident grids, each uploaded, advanced one step and downloaded
               (PPM.step_host_pipelined): the slabs of grid s+1 go up while the slabs of grid s come down."""
    ncell = n ** 3
    host_a = torch.empty((NF, n, n, n), dtype=torch.float32, pin_memory=True)
    host_out = torch.empty((NF, n, n, n), dtype=torch.float32, pin_memory=True)
    host_out2 = torch.empty((NF, n, n, n), dtype=torch.float32, pin_memory=True) if g2 is not None else None
    g.get_state(out=host_a)
    g.set_state(host_a); do_step(dt, 0); g.get_state(out=host_out)      # warm-up
    barrier()
    t0 = time.perf_counter()
    for s in range(Ke):
        g.set_state(host_a)
        do_step(dt, 0 if s % 2 == 0 else 5)
        g.get_state(out=host_out)       # synchronises
    torch.cuda.synchronize()
    serial = (time.perf_counter() - t0) * 1e3 / Ke
    res = {"serial_ms": serial, "steps": Ke, "bytes": NF * ncell * 4}
    try:
        # what the link itself does with this traffic: the grid up and down at once, plain copies on two streams, nothing else
        dev_t = torch.empty((2, NF, n, n, n), dtype=torch.float32, device=g.device)
        s_up, s_dn = torch.cuda.Stream(g.device), torch.cuda.Stream(g.device)
        dev_t[1].copy_(host_out)                       # host_out keeps its values (it seeds the second input grid below)
        for rep in range(2):
            torch.cuda.synchronize()
            t0 = time.perf_counter()
            with torch.cuda.stream(s_up):
                dev_t[0].copy_(host_a, non_blocking=True)
            with torch.cuda.stream(s_dn):
                host_out.copy_(dev_t[1], non_blocking=True)
            torch.cuda.synchronize()
            res["link_duplex_ms"] = (time.perf_counter() - t0) * 1e3
        del dev_t
    except Exception as ex:
        res["link_error"] = str(ex)[:200]
    try:
        host_b = torch.empty((NF, n, n, n), dtype=torch.float32, pin_memory=True)
        host_b.copy_(host_out)
        ins = [host_a, host_b]
        g.step_host_pipelined([host_a], [host_out], dt, [0], step=do_step)            # warm-up (allocates the staging slabs)
        barrier()
        Kp = max(Ke, 4)
        t0 = time.perf_counter()
        g.step_host_pipelined([ins[s % 2] for s in range(Kp)], [host_out] * Kp, dt, [0 if s % 2 == 0 else 5 for s in range(Kp)],
                              step=do_step)
        torch.cuda.synchronize()
        res["pipelined_ms"] = (time.perf_counter() - t0) * 1e3 / Kp
        res["pipelined_steps"] = Kp
        # two contexts on two streams, each fed with every other grid: while one computes and downloads, the other uploads
        if g2 is not None:
            try:
                st2 = g2.step if do_step == g.step else g2.advect
                g2.step_host_pipelined([host_b], [host_out], dt, [0], step=st2)               # warm-up (staging slabs)
                barrier()
                seq = [(ins[s % 2], 0 if s % 2 == 0 else 5) for s in range(2 * Kp)]
                t0 = time.perf_counter()
                g.step_host_pipelined([x for x, _ in seq[0::2]], [host_out] * Kp, dt, [o for _, o in seq[0::2]], step=do_step, wait=False)
                g2.step_host_pipelined([x for x, _ in seq[1::2]], [host_out2] * Kp, dt, [o for _, o in seq[1::2]], step=st2, wait=False)
                g.finish_host_pipelined(); g2.finish_host_pipelined()
                torch.cuda.synchronize()
                res["pipelined2_ms"] = (time.perf_counter() - t0) * 1e3 / (2 * Kp)
                res["pipelined2_steps"] = 2 * Kp
            except Exception as ex:
                res["pipelined2_error"] = str(ex)[:200]
        del host_b
    except Exception as ex:
        res["pipelined_error"] = str(ex)[:200]
    del host_a, host_out
    return res


def run_gpu(args):
    ws, rank, lr = _dist()
    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device; the PPM+PPB path has no CPU fallback")
    torch.cuda.set_device(lr)
    dev = torch.device("cuda", lr)
    if ws > 1:
        import torch.distributed as dist
        dist.init_process_group("nccl", device_id=dev)

    def barrier():
        if ws > 1:
            dist.barrier()
        torch.cuda.synchronize()

    K = args.steps
    reps = args.reps if args.reps else (3 if args.workload == 5 else 5)
    r = _bench_grid(args, args.workload, dev, lr, ws, barrier, K, reps, not args.no_e2e)
    # second target grid in the same run: config 5 (1024^3, its 5 steps x 3 repetitions) when the headline is config 4
    also = None
    want_also = (args.workload == 4 and not args.no_also and not args.advect and not args.direct and not args.two_fluid
                 and torch.cuda.get_device_properties(dev).total_memory > 150e9)
    if want_also:
        try:
            also = _bench_grid(args, 5, dev, lr, ws, barrier, 5, 3, False)
        except Exception as ex:
            also = {"error": str(ex)[:200]}

    # ---- reduce over ranks (max of the per-rank times) ----
    def med(x):
        return float(np.median(x))
    ms = med(r["ms_reps"])
    ms_cfl = med(r["ms_cfl"])
    e2e = r["e2e"]
    if e2e and e2e.get("pipelined2_ms") and e2e["pipelined2_ms"] < e2e.get("pipelined_ms", 1e30):
        e2e["pipelined_ms_1ctx"] = e2e.get("pipelined_ms")
        e2e["pipelined_ms"], e2e["pipelined_steps"], e2e["two_ctx"] = e2e["pipelined2_ms"], e2e["pipelined2_steps"], True
    vals = [ms, ms_cfl, (e2e or {}).get("serial_ms", 0.0), (e2e or {}).get("pipelined_ms", 0.0),
            med(also["ms_reps"]) if also and "ms_reps" in also else 0.0]
    if ws > 1:
        vals = max_over_ranks(vals, ws, dev)
    ms, ms_cfl, e_ser, e_pipe, ms_also = vals
    if rank != 0:
        if ws > 1:
            dist.destroy_process_group()
        return 0

    peak, peak_kind = _peaks()
    w, n = r["w"], r["n"]
    ncell = n ** 3
    fp32_peak, fp32_kind = (r["fp32"], "measured: FFMA micro-benchmark in this run (ppm_measure_fp32_peak)") if r["fp32"] else \
        (FP32_NOMINAL_TFLOPS, "nominal: SMs x 128 lanes x 2 x max SM clock")
    line = {
        "metric": METRIC, "value": aggregate_value(ncell, K, ms, ws), "unit": UNIT, "n_gpus": ws, "steps": K, "warmup": r["warmup"],
        "ms_per_step": ms / K, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
        "dtype": "f32", "data": "synthetic",
        "config": {"workload": "%s %d^3, %s, dt fixed at 0.7*CFL dt, sweep order xyz/zyx alternating" % (w.name, n, _geometry(w)),
                   "cells_per_gpu": ncell, "l2": "inputs (%.1f GB state) larger than the 126 MB L2" % (15 * ncell * 4 / 1e9),
                   "parallelism": "replicas only (1 grid per GPU)", "chunk": args.chunk,
                   "flatten": "3-D detector field" if args.flatten3d else "1-D per sweep (baseline scheme)",
                   "eos": "two-fluid: gamma 1.4 (tracked, FV) / 5/3 (ppm_set_two_fluid; reading R25)" if args.two_fluid else "one ideal gas",
                   "geometry": "star inside the confining sphere inscribed in the cube (ppm_set_sphere; PAPER.md L69): cell-updates count ALL cells of the cube, 52 % of which are fluid" if args.sphere else "reflecting cube",
                   "step": "PPB-only advection (ppm_advect; 84 B/cell/sweep algorithmic and moved: the hydro fields stay in their buffer)" if args.advect else "full PPM+PPB (ppm_step, CFL max-reduction fused into the last sweep)",
                   "fv_shortcut": "on (library default): the PPB remap is skipped where FV is uniform under a whole warp — same values; 'without_fv_shortcut' is the same run with it off",
                   "timing": "median of %d repetitions of the %d-step region (CUDA events on the library's stream)" % (len(r["ms_reps"]), K)},
        "repetitions_ms_per_step": [x / K for x in r["ms_reps"]],
        "roofline": _roofline(n, ms / K, args.advect, peak, peak_kind, fp32_peak, fp32_kind),
        "clocks": r["clocks"], "gpu_launches": int(r["launches"]),
        "without_fv_shortcut": ({"value": aggregate_value(ncell, K, med(r["ms_noskip"]), ws), "unit": UNIT, "ms_per_step": med(r["ms_noskip"]) / K,
                                 "roofline_frac": BYTES_PER_CELL_SWEEP * ncell * 3 * K / (med(r["ms_noskip"]) * 1e-3) / 1e9 / peak,
                                 "note": "PPM_OPT_FV_SHORTCUT = 0: the PPB remap runs in every cell, also where FV is uniform under a whole warp (this rank's time); same values"}
                                if r["ms_noskip"] else None),
        "with_cfl_dt": {"value": aggregate_value(ncell, K, ms_cfl, ws), "unit": UNIT, "ms_per_step": ms_cfl / K,
                        "note": "ppm_cfl_dt before every step: the maximum is reduced inside the previous step's last sweep, so this is a 4-byte read + host sync"},
    }
    if e2e and "serial_ms" in e2e:
        best = e_pipe if e_pipe > 0 else e_ser
        line["e2e"] = {"value": ws * ncell / (best * 1e-3), "unit": UNIT, "h2d_bytes_per_step": e2e["bytes"],
                       "d2h_bytes_per_step": e2e["bytes"], "steps": e2e.get("pipelined_steps", e2e["steps"]), "ms_per_step": best,
                       "mode": (("independent host-resident grids, one step each, dealt to TWO contexts on two streams (PPM.step_host_pipelined, wait=False): "
                                 "while one context computes and downloads, the other uploads; within a context the upload slabs of its next grid overlap "
                                 "the download slabs of the current one") if e2e.get("two_ctx") else
                                ("independent host-resident grids, one step each: the upload slabs of grid s+1 overlap the download slabs of grid s "
                                 "(PPM.step_host_pipelined, two copy streams)")) if e_pipe > 0 else "serial: set_state(host), step, get_state(host) on one stream",
                       "one_context_pipelined_ms_per_step": e2e.get("pipelined2_ms") and e2e.get("pipelined_ms_1ctx"),
                       "serial_ms_per_step": e_ser,
                       "pcie_floor_ms": e2e["bytes"] / 55e9 * 1e3,
                       "link_duplex_ms": e2e.get("link_duplex_ms"),   # measured here: the same bytes up and down at once, copies only
                       "note": e2e.get("pipelined_error")}
    else:
        line["e2e"] = {"value": None, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0,
                       "note": (e2e or {}).get("error", "skipped")}
    if also and "ms_reps" in also:
        n5 = also["n"]
        fp5 = (also["fp32"], fp32_kind) if also["fp32"] else (fp32_peak, fp32_kind)
        line["also"] = {"workload": "%s %d^3 (BASELINE.json configs[4]: its 5 steps, %d repetitions, same process)" % (also["w"].name, n5, len(also["ms_reps"])),
                        "value": aggregate_value(n5 ** 3, 5, ms_also, ws), "unit": UNIT, "steps": 5, "ms_per_step": ms_also / 5,
                        "repetitions_ms_per_step": [x / 5 for x in also["ms_reps"]],
                        "roofline": _roofline(n5, ms_also / 5, False, peak, peak_kind, fp5[0], fp5[1]),
                        "clocks": also["clocks"], "gpu_launches": int(also["launches"]),
                        "with_cfl_dt_ms_per_step": med(also["ms_cfl"]) / 5,
                        "without_fv_shortcut_ms_per_step": (med(also["ms_noskip"]) / 5 if also["ms_noskip"] else None)}
    elif also:
        line["also"] = also
    if ws == 1 and not args.no_cpu_baseline:
        line["cpu_baseline"] = _cpu_baseline(w)
    print(json.dumps(line))
    if ws > 1:
        dist.destroy_process_group()
    return 0


def run_decomposed(args):
    """--decompose px,py,pz: ONE global grid (the workload) cut into px*py*pz sub-domains, a brick layer
    exchanged with the face neighbours before every sweep.  Under torchrun with px*py*pz ranks: one sub-domain per GPU, NCCL
    send/recv over NVLink ("strong" scaling: the total work is fixed).  In a single process: all sub-domains on this GPU
    (LocalCluster, device copies) — what the decomposition itself costs (packing, copies, shorter pencils), measured where only
    one GPU is to be had."""
    from paper_1810_13416_b200.decomposition import BrickDecomposition, DecomposedPPM, LocalCluster
    ws, rank, lr = _dist()
    procs = tuple(int(v) for v in args.decompose.split(","))
    torch.cuda.set_device(lr)
    dev = torch.device("cuda", lr)
    w = W.make(args.workload)
    n = w.n
    d = BrickDecomposition((n, n, n), procs, w.bc)
    if ws > 1:
        import torch.distributed as dist
        assert ws == d.size, "--decompose %s needs %d ranks" % (args.decompose, d.size)
        dist.init_process_group("nccl", device_id=dev)

    def barrier():
        if ws > 1:
            dist.barrier()
        torch.cuda.synchronize()

    if ws > 1:
        g = DecomposedPPM(d, rank, w.dx, w.gamma, w.grav, w.rho_floor, w.p_floor, dev)
        parts = [g]
    else:
        g = LocalCluster(d, w.dx, w.gamma, w.grav, w.rho_floor, w.p_floor, dev)
        parts = g.parts
    for p in parts:                                   # every sub-domain generates its own box of the synthetic input
        o, ln = p.org, d.local_n()
        for z0 in range(0, ln[2], 32):
            z1 = min(ln[2], z0 + 32)
            p.ppm.set_state(w.fields((o[0], o[1], o[2] + z0), (o[0] + ln[0], o[1] + ln[1], o[2] + z1), device=dev), z0=z0)
    dt = 0.7 * g.cfl_dt(w.cfl)
    K, Wm = args.steps, max(args.warmup, 3)
    for s in range(Wm):
        g.step(dt, 0 if s % 2 == 0 else 5)
    barrier()
    clk = _Clocks(lr)
    reps = args.reps if args.reps else 5
    ms_reps = []
    b0 = sum(p.halo_bytes for p in parts)
    for r in range(reps):
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        barrier()
        e0.record(parts[0].ppm.stream)
        for s in range(K):
            g.step(dt, 0 if s % 2 == 0 else 5)
        e1.record(parts[0].ppm.stream)
        barrier()
        ms_reps.append(e0.elapsed_time(e1))
    halo = (sum(p.halo_bytes for p in parts) - b0) / (reps * K)
    clocks = clk.stop()
    for p in parts:
        p.ppm.sync()
    ms = float(np.median(ms_reps))
    vals = max_over_ranks([ms, halo], ws, dev) if ws > 1 else [ms, halo]
    if rank == 0:
        peak, peak_kind = _peaks()
        line = {"metric": METRIC, "value": n ** 3 * K / (vals[0] * 1e-3), "unit": UNIT, "n_gpus": ws, "steps": K, "warmup": Wm,
                "ms_per_step": vals[0] / K, "higher_is_better": True, "scaling": "strong", "vs_baseline": None, "dtype": "f32", "data": "synthetic",
                "config": {"workload": "%s %d^3 as ONE grid cut into %s sub-domains of %s cells" % (w.name, n, "x".join(map(str, procs)), "x".join(map(str, d.local_n()))),
                           "parallelism": ("brick decomposition, one sub-domain per GPU, NCCL send/recv of one brick layer per face before each sweep" if ws > 1 else
                                           "brick decomposition, all %d sub-domains on ONE GPU (device copies for the messages)" % d.size),
                           "halo_bytes_per_step_per_rank_max": vals[1],
                           "timing": "median of %d repetitions of the %d-step region (CUDA events)" % (reps, K)},
                "repetitions_ms_per_step": [x / K for x in ms_reps], "clocks": clocks,
                "roofline": {"bound": "hbm", "achieved": BYTES_PER_CELL_SWEEP * n ** 3 * 3 * K / (vals[0] * 1e-3) / 1e9 / ws, "peak": peak, "unit": "GB/s",
                             "frac": BYTES_PER_CELL_SWEEP * n ** 3 * 3 * K / (vals[0] * 1e-3) / 1e9 / ws / peak, "traffic": None, "peak_kind": "of " + peak_kind,
                             "note": "per GPU: sweeps + packing + exchange"},
                "gpu_launches": int(sum(p.ppm.launch_count() for p in parts))}
        print(json.dumps(line))
    g.close()
    if ws > 1:
        dist.destroy_process_group()
    return 0


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=10)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--reps", type=int, default=0, help="repetitions of the K-step region (default 5; 3 at 1024^3)")
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--workload", type=int, default=4, help="BASELINE.json config number (4 = 512^3, 5 = 1024^3)")
    ap.add_argument("--chunk", type=int, default=0)
    ap.add_argument("--advect", action="store_true", help="time PPB-only steps (ppm_advect, SURVEY 8(f) NEXT-2) instead of full PPM+PPB steps")
    ap.add_argument("--flatten3d", action="store_true", help="fully 3-D shock-flattening mode (SURVEY 8(f) NEXT-1): one more light kernel per step")
    ap.add_argument("--sphere", action="store_true", help="the paper's run geometry (SURVEY 8(f) NEXT-3): confining sphere inscribed in the cube")
    ap.add_argument("--two-fluid", action="store_true", help="two-fluid equation of state (SURVEY 8(f) NEXT-4): the tracked fluid has gamma = 1.4")
    ap.add_argument("--decompose", default="", help="px,py,pz: the workload as ONE grid cut into sub-domains with halo exchange (SURVEY 8(f) NEXT-4); under torchrun with px*py*pz ranks one sub-domain per GPU, else all on this GPU")
    ap.add_argument("--direct", action="store_true", help="direct global-memory sweep path instead of the bulk-staged one")
    ap.add_argument("--e2e-steps", type=int, default=2)
    ap.add_argument("--ref-side", type=int, default=128, help="side of the oracle's sample window (--impl reference)")
    ap.add_argument("--no-e2e", action="store_true")
    ap.add_argument("--no-also", action="store_true", help="skip the 1024^3 entry of the default run")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    args = ap.parse_args()
    if args.impl == "reference":
        return run_reference(args)
    if args.decompose:
        return run_decomposed(args)
    return run_gpu(args)


if __name__ == "__main__":
    sys.exit(main())
