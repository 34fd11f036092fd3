#!/usr/bin/env python
"""bench.py — cell-updates/s of the fused PPM+PPB timestep on B200 (BASELINE.json metric).

  python bench.py [--gpus N] [--steps K] [--warmup W] [--workload 4|5|...] [--impl reference]

A "step" is one ppm_step = the whole hot path (three fused hydro+PPB sweeps) over the
whole synthetic grid.  value = cells * K / device time (CUDA events, max over ranks), inputs resident in
HBM.  e2e = the same metric through the C ABI with pinned HOST buffers: ppm_set_state(host) + ppm_step +
ppm_get_state(host) inside the timed region.  Multi-GPU: the path is "replicas only": each
rank advances its own grid, no data-path collective; value sums the ranks' cells ("weak" scaling).

--impl reference times the fp64 CPU oracle (as it stands) on a bounded window of the same workload.
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
BYTES_PER_CELL_SWEEP_ADVECT = 84.0   # PPB-only sweep: 1 velocity + 10 coefficients read, 10 written (it moves 120: hydro copied through)
FLOPS_PER_CELL_SWEEP = 1307.0     # operation count of the oracle's sweep body, FMA = 2
FP32_PEAK_TFLOPS = 148 * 128 * 2 * 1.965e9 / 1e12   # SMs x lanes x FMA x max SM clock (B200_PROFILING.md)
# dram__bytes_read.sum + dram__bytes_write.sum per sweep launch from the committed `ncu --set full` capture
# (profiles/), keyed by cells per side; None where no capture exists.
NCU_TRAFFIC_BYTES = {512: 16.099e9}      # profiles/r1h_sweeps_ncu_full.md: 8.089 GB read + 8.010 GB written per launch


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


def _load_state(g, w, nzs):
    n = w.n
    for z0 in range(0, n, nzs):
        z1 = min(n, z0 + nzs)
        g.set_state(w.fields((0, 0, z0), (n, n, z1), device=g.device), z0=z0)


def _sample_window(w, side):
    """central window of the workload used for the oracle timings"""
    side = min(side, w.n)
    lo = [(w.n - side) // 2] * 3
    hi = [lo[0] + side] * 3
    bc = [w.bc[k] if side == w.n else 2 for k in range(6)]
    return lo, hi, bc


def _time_oracle(w, side, steps, warmup):
    from oracle import binding as ob          # bench.py's cpu_baseline / reference legs may use oracle/
    lo, hi, bc = _sample_window(w, side)
    f = w.fields(lo, hi).numpy()
    o = ob.Oracle(hi[0] - lo[0], hi[1] - lo[1], hi[2] - lo[2], w.dx, w.gamma, bc, w.grav, org=lo,
                  rho_floor=w.rho_floor, p_floor=w.p_floor)
    o.set_state(f)
    dt = 0.5 * o.cfl_dt(w.cfl)
    for s in range(warmup):
        o.step(dt, 0 if s % 2 == 0 else 5)
    t0 = time.perf_counter()
    for s in range(steps):
        o.step(dt, 0 if s % 2 == 0 else 5)
    t = time.perf_counter() - t0
    cells = (hi[0] - lo[0]) ** 3
    return cells * steps / t, t / steps, ob.num_threads(), "central %d^3 window of %s, %d steps" % (hi[0] - lo[0], w.name, steps)


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


def run_gpu(args):
    ws, rank, lr = _dist()
    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device; the PPM+PPB path has no CPU fallback")
    torch.cuda.set_device(lr)
    dev = torch.device("cuda", lr)
    if ws > 1:
        import torch.distributed as dist
        dist.init_process_group("nccl", device_id=dev)
    from paper_1810_13416_b200.binding import PPM, NF

    w = W.make(args.workload)
    n = w.n
    ncell = n ** 3
    g = PPM.from_workload(w, device=dev)
    if args.chunk:
        g.set_chunk(args.chunk)
    if args.direct:
        from paper_1810_13416_b200.binding import OPT_IO_PATH
        g.set_option(OPT_IO_PATH, 1)
    if args.flatten3d:
        from paper_1810_13416_b200.binding import OPT_FLATTEN3D
        g.set_option(OPT_FLATTEN3D, 1)
    _load_state(g, w, 8 if n >= 1024 else 32)
    dt = 0.7 * g.cfl_dt(w.cfl)       # fixed for the run: no host sync inside the timed region
    do_step = g.advect if args.advect else g.step

    def barrier():
        if ws > 1:
            dist.barrier()
        torch.cuda.synchronize()

    K, Wm = args.steps, max(args.warmup, 3)
    for s in range(Wm):
        do_step(dt, 0 if s % 2 == 0 else 5)
    barrier()
    clk = _Clocks(lr)
    l0 = g.launch_count()
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    barrier()
    e0.record(g.stream)
    for s in range(K):
        do_step(dt, 0 if s % 2 == 0 else 5)
    e1.record(g.stream)
    barrier()
    ms = e0.elapsed_time(e1)
    launches = g.launch_count() - l0
    clocks = clk.stop()
    g.sync()                         # raises if the state flag (NaN / floor) was set

    # ---- the same K steps with ppm_cfl_dt before each one (SURVEY 8(d) "also report with ppm_cfl_dt per step
    # included"): one more reduction kernel and one host sync per step ----
    e2, e3 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    barrier()
    e2.record(g.stream)
    for s in range(K):
        do_step(0.7 * g.cfl_dt(w.cfl), 0 if s % 2 == 0 else 5)
    e3.record(g.stream)
    barrier()
    ms_cfl = e2.elapsed_time(e3)
    if ws > 1:
        ms_cfl = max_over_ranks([ms_cfl], ws, dev)[0]

    # ---- e2e: host buffers through the C ABI, copies inside the timed region ----
    e2e = None
    if not args.no_e2e:
        try:
            Ke = args.e2e_steps
            host_in = torch.empty((NF, n, n, n), dtype=torch.float32, pin_memory=True)
            host_out = torch.empty((NF, n, n, n), dtype=torch.float32, pin_memory=True)
            g.get_state(out=host_in)
            g.set_state(host_in); do_step(dt, 0); g.get_state(out=host_out)      # warm-up
            barrier()
            t0 = time.perf_counter()
            for s in range(Ke):
                g.set_state(host_in)
                do_step(dt, 0 if s % 2 == 0 else 5)
                g.get_state(out=host_out)       # synchronises
                host_in, host_out = host_out, host_in
            torch.cuda.synchronize()
            te = time.perf_counter() - t0
            e2e = {"ms": te * 1e3 / Ke, "steps": Ke, "bytes": NF * ncell * 4}
            del host_in, host_out
        except Exception as ex:                                                  # e.g. not enough pinned host memory
            e2e = {"error": str(ex)[:200]}

    # ---- reduce over ranks ----
    if ws > 1:
        red = max_over_ranks([ms, e2e["ms"] if e2e and "ms" in e2e else 0.0], ws, dev)
        ms = red[0]
        if e2e and "ms" in e2e:
            e2e["ms"] = red[1]
    if rank != 0:
        if ws > 1:
            dist.destroy_process_group()
        return 0

    peak, peak_kind = _peaks()
    value = aggregate_value(ncell, K, ms, ws)
    # the dominant kernel = the 3 sweep launches of every step (in --flatten3d mode the light detector kernel's time
    # is charged to them: conservative)
    per_launch_s = ms * 1e-3 / (3 * K)
    achieved = (BYTES_PER_CELL_SWEEP_ADVECT if args.advect else BYTES_PER_CELL_SWEEP) * ncell / per_launch_s / 1e9
    flops_cs = 478.0 if args.advect else FLOPS_PER_CELL_SWEEP     # PPB-only: P2 13 + P1/P3/P4 460 + face masses 5
    alu = flops_cs * ncell / per_launch_s / 1e12
    line = {
        "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": ws, "steps": K, "warmup": Wm,
        "ms_per_step": ms / K, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
        "dtype": "f32", "data": "synthetic",
        "config": {"workload": "%s %d^3, %s, dt fixed at 0.7*CFL dt, sweep order xyz/zyx alternating" % (w.name, n, "reflecting walls + radial gravity" if w.grav else "periodic"),
                   "cells_per_gpu": ncell, "l2": "inputs (%.1f GB state) larger than the 126 MB L2" % (NF * ncell * 4 / 1e9),
                   "parallelism": "replicas only (1 grid per GPU)", "chunk": args.chunk,
                   "flatten": "3-D detector field" if args.flatten3d else "1-D per sweep (baseline scheme)",
                   "step": "PPB-only advection (ppm_advect; 84 B/cell/sweep algorithmic, 120 moved)" if args.advect else "full PPM+PPB (ppm_step)"},
        "roofline": {"bound": "hbm", "achieved": achieved, "peak": peak, "unit": "GB/s", "frac": achieved / peak,
                     "traffic": NCU_TRAFFIC_BYTES.get(n), "peak_kind": "of " + peak_kind,
                     "kernel": ("ppm_advect_bulk_kernel" if args.advect else "ppm_sweep_bulk_kernel") + " (3 launches per step; every launch moves 120 B/cell)",
                     "alu": {"achieved": alu, "peak": FP32_PEAK_TFLOPS, "unit": "TFLOP/s", "frac": alu / FP32_PEAK_TFLOPS,
                             "flops_per_cell_sweep": flops_cs}},
        "clocks": clocks, "gpu_launches": int(launches),
        "with_cfl_dt": {"value": aggregate_value(ncell, K, ms_cfl, ws), "unit": UNIT, "ms_per_step": ms_cfl / K,
                        "note": "ppm_cfl_dt (max-reduction kernel + host sync) before every step"},
    }
    if e2e and "ms" in e2e:
        line["e2e"] = {"value": ws * ncell / (e2e["ms"] * 1e-3), "unit": UNIT, "h2d_bytes_per_step": e2e["bytes"],
                       "d2h_bytes_per_step": e2e["bytes"], "steps": e2e["steps"], "ms_per_step": e2e["ms"]}
    else:
        line["e2e"] = {"value": None, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0,
                       "note": (e2e or {}).get("error", "skipped")}
    if ws == 1 and not args.no_cpu_baseline:
        val, _, cores, sample = _time_oracle(w, args.ref_side, 2, 0)
        line["cpu_baseline"] = {"value": val, "unit": UNIT, "cores": cores, "kind": "oracle", "sample": sample}
    print(json.dumps(line))
    if ws > 1:
        dist.destroy_process_group()
    return 0


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=10)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--workload", type=int, default=4, help="BASELINE.json config number (4 = 512^3, 5 = 1024^3)")
    ap.add_argument("--chunk", type=int, default=0)
    ap.add_argument("--advect", action="store_true", help="time PPB-only steps (ppm_advect, SURVEY 8(f) NEXT-2) instead of full PPM+PPB steps")
    ap.add_argument("--flatten3d", action="store_true", help="fully 3-D shock-flattening mode (SURVEY 8(f) NEXT-1): one more light kernel per step")
    ap.add_argument("--direct", action="store_true", help="direct global-memory sweep path instead of the bulk-staged one")
    ap.add_argument("--e2e-steps", type=int, default=2)
    ap.add_argument("--ref-side", type=int, default=128, help="side of the oracle's sample window")
    ap.add_argument("--no-e2e", action="store_true")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    args = ap.parse_args()
    if args.impl == "reference":
        return run_reference(args)
    return run_gpu(args)


if __name__ == "__main__":
    sys.exit(main())
