#!/usr/bin/env python
"""bench.py -- throughput of the RK4 hot path on B200 (BASELINE.json metric: grid-cell RK4 steps per second).

    python bench.py [--gpus N] [--steps K] [--warmup W] [--workload NAME] [--variant V] [--impl reference]

A "step" is one RK4 step (all four stages, plus noise where the workload has it) over the whole grid /
ensemble.  `value` times K steps with the state resident in HBM (CUDA events on the launching stream,
barrier + synchronize on both sides, max over ranks).  `e2e` times the same metric through the C ABI with
HOST buffers: every step uploads psi from pinned host memory, runs one RK4 step and downloads psi.
The path does not shard (replicas only): with --gpus N each rank steps an independent
replica of the workload and `value` is the sum.  Prints ONE JSON line on rank 0.
"""
import argparse
import json
import os
import statistics
import subprocess
import sys
import threading
import time

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

import numpy as np  # noqa: E402

METRIC = "grid-cell RK4 steps/sec"
UNIT = "Gcell*step/s"

# Compulsory (infinite-cache) bytes per cell-step, fp32 (fp64: x2); DESIGN.md section 6.
COMPULSORY_BYTES = {"scalar": 20, "reservoir": 28, "spinor": 32, "spinor_reservoir": 52}


def build_workload(name):
    from paper_2411_18341_b200 import workloads as wl
    table = {
        "cfg1": lambda: wl.cfg1(),
        "cfg2_1024_c32": lambda: wl.cfg2(1024, "c32"), "cfg2_1024_c64": lambda: wl.cfg2(1024, "c64"),
        "cfg2_4096_c32": lambda: wl.cfg2(4096, "c32"), "cfg2_4096_c64": lambda: wl.cfg2(4096, "c64"),
        "cfg3_4096_c32": lambda: wl.cfg3(4096, "c32"),
        "cfg4_16384_c32": lambda: wl.cfg4(16384, "c32"), "cfg4_8192_c32": lambda: wl.cfg4(8192, "c32"),
        "cfg5_512x256_c32": lambda: wl.cfg5(256, 512, "c32"),
        # small-grid regime: one 64^2 grid, and an ensemble of 64^2 grids
        "cfg2_64_c32": lambda: wl.cfg2(64, "c32"), "cfg5_512x64_c32": lambda: wl.cfg5(64, 512, "c32"),
        "cfg5_512x64_c64": lambda: wl.cfg5(64, 512, "c64"),
    }
    if name not in table:
        raise SystemExit(f"unknown workload {name}; choose from {sorted(table)}")
    return table[name]()


def algo_bytes_per_cell_step(w, variant, steps_per_launch=1):
    """Algorithmic HBM bytes per cell-step of variant STAGE, counted array by array.

    Per complex component: s1 R psi, W y2; s2 R y2, psi, W y3, acc; s3 R y3, psi, acc, W y4, acc;
    s4 R y4, acc, W psi = 14 complex transfers.  Per reservoir: s1 R n, W n2; s2 R n2, n, W n3, nacc;
    s3 R n3, n, nacc, W n4, nacc; s4 R n4, nacc, W n = 14 real transfers.  V, P: one real read per stage."""
    rb = 8 if w.prec == "c64" else 4
    ncomp = 2 if w.model.startswith("spinor") else 1
    res = w.model.endswith("reservoir")
    if variant == 4:
        # variant RESIDENT: the same arrays once per LAUNCH (all steps of the call run on chip)
        return algo_bytes_per_cell_step(w, 3) / max(1, steps_per_launch)
    if variant == 3:
        # variant STEP: every state array is read once and written once per step; V, P read once
        b = ncomp * 2 * 2 * rb + (ncomp * 2 * rb if res else 0)
        b += rb if w.V is not None else 0
        b += rb if (res and w.P is not None) else 0
        return b
    b = ncomp * 14 * 2 * rb
    if res:
        b += ncomp * 14 * rb
        if w.P is not None:
            b += 4 * rb
        if w.noise:
            b += ncomp * rb                                 # n_t re-read for sigma (Eq. 22)
    if w.V is not None:
        b += 4 * rb
    return b


def algo_flops_per_cell_step(w):
    """Floating-point operations the method itself asks for per cell-step (counted from the
    formulas of section 2, an FMA = 2): per stage and component the derivative costs 33 (Laplacian 18, density 4,
    potential 3, K 8), +9 with a reservoir (g_r n 2, gain 3, K_n 4), +36 in a spinor (cross density 6, TE-TM 30);
    the fused RK sums cost 28 per component (+14 per reservoir).  The Philox/Box-Muller work of the noise is not counted."""
    ncomp = 2 if w.model.startswith("spinor") else 1
    res = w.model.endswith("reservoir")
    per_stage = 33 + (9 if res else 0) + (36 if ncomp == 2 else 0)
    return ncomp * (4 * per_stage + 28 + (14 if res else 0))


# Plain-ALU peak (no tensor cores: the stencil is not a contraction): 148 SMs x 128 FP32 (64 FP64) lanes x 2 flop x
# 1.965 GHz (B200_PROFILING.md unit counts and clocks.max.sm); DESIGN.md section 6.
ALU_PEAK_TFLOPS = {"c32": 148 * 128 * 2 * 1.965e9 / 1e12, "c64": 148 * 64 * 2 * 1.965e9 / 1e12}


class ClockSampler:
    """Samples nvidia-smi clocks and throttle reasons while the timed region runs."""
    Q = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,clocks_event_reasons.hw_thermal_slowdown,"
         "clocks_event_reasons.sw_thermal_slowdown,clocks_event_reasons.sw_power_cap")

    def __init__(self, index):
        self.rows, self.proc, self.index = [], None, index

    def start(self):
        try:
            self.proc = subprocess.Popen(["nvidia-smi", f"--query-gpu={self.Q}", "--format=csv,noheader,nounits", "-lms", "100",
                                          "-i", str(self.index)], stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
            self.t = threading.Thread(target=self._read, daemon=True)
            self.t.start()
        except Exception:
            self.proc = None

    def _read(self):
        for line in self.proc.stdout:
            self.rows.append((time.time(), line.strip()))

    def stop(self, t0, t1):
        if self.proc is None:
            return None
        time.sleep(0.15)
        self.proc.terminate()
        try:
            self.proc.wait(timeout=2)
        except Exception:
            self.proc.kill()
        sm, mx, reasons, pw = [], [], set(), []
        rows = [r for r in self.rows if t0 <= r[0] <= t1 + 0.2] or self.rows[-3:]
        for _, line in rows:
            p = [v.strip() for v in line.split(",")]
            try:
                sm.append(float(p[0])); mx.append(float(p[1])); pw.append(float(p[2]))
            except Exception:
                continue
            for name, v in zip(("hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"), p[3:7]):
                if v.lower().startswith("active"):
                    reasons.add(name)
        if not sm:
            return None
        return {"sm_mhz": statistics.median(sm), "sm_max_mhz": max(mx), "power_w_max": max(pw), "samples": len(sm),
                "reasons": sorted(reasons)}


def measured_peaks():
    path = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(path):
        try:
            return float(json.load(open(path))["hbm_gbs"]), "measured (MEASURED_PEAKS.json hbm_gbs)"
        except Exception:
            pass
    return 6650.0, "fallback (B200_PROFILING.md 6.65 TB/s)"


def max_over_ranks(x, world, device="cuda"):
    """A time is the slowest rank's (the contract: device time, max over ranks)."""
    if world <= 1:
        return float(x)
    import torch
    import torch.distributed as dist
    t = torch.tensor([float(x)], device=device, dtype=torch.float64)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())


def whole_job_value(world, cells, steps, ms):
    """Replicas only: every rank steps its own copy, the job's cell-steps add up."""
    return world * cells * steps / (ms * 1e-3) / 1e9


def oracle_from_workload(w, ny=None):
    """The oracle as it stands on (a row-slab sample of) the workload."""
    import oracle as orc
    ny = w.ny if ny is None else ny
    o = orc.Oracle(w.nx, ny, w.dx, w.dy, orc.make_params(**w.params), model=w.model, batch=1, prec32=(w.prec == "c32"),
                   noise=w.noise, seed=w.seed, V=None if w.V is None else w.V[:ny].astype(np.float64),
                   P=None if w.P is None else w.P[:ny].astype(np.float64))
    for name, arr in w.fields.items():
        o.set_field(name, arr[:1, :ny])
    return o


def run_reference(args):
    """--impl reference: the CPU oracle, as it stands, on a bounded sample of the same workload."""
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    w = build_workload(args.workload)
    # bounded sample: ~60 s of single-thread oracle work (~7 Mcell*step/s) over the whole run
    target_cells = int(4.0e8 / max(1, args.steps + args.warmup))
    ny = max(8, min(w.ny, target_cells // w.nx))
    o = oracle_from_workload(w, ny)
    for _ in range(args.warmup):
        o.step_rk4(1)
    t0 = time.perf_counter()
    for _ in range(args.steps):
        o.step_rk4(1)
    dt = time.perf_counter() - t0
    cells = w.nx * ny
    val = cells * args.steps / dt / 1e9
    sample = f"{w.nx}x{ny} row slab of realisation 0 (periodic), 1 RK4 step per bench step"
    print(json.dumps({
        "impl": "reference", "metric": METRIC, "value": val, "unit": UNIT, "n_gpus": args.gpus, "steps": args.steps,
        "warmup": args.warmup, "ms_per_step": dt / args.steps * 1e3, "higher_is_better": True, "scaling": "weak",
        "vs_baseline": None, "dtype": "f64", "data": "synthetic",
        "config": {"workload": args.workload, "sample": sample},
        "cpu_baseline": {"value": val, "unit": UNIT, "cores": 1, "kind": "oracle", "sample": sample},
        "e2e": {"value": val, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
    }))


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=2000)
    ap.add_argument("--warmup", type=int, default=50)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--workload", default="cfg2_4096_c32")
    ap.add_argument("--variant", type=int, default=0)
    ap.add_argument("--tune", default="", help="comma separated key=value passed to phx_set_tuning")
    ap.add_argument("--e2e-steps", type=int, default=20)
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-stage-leg", action="store_true", help="skip the extra timing of variant STAGE")
    args = ap.parse_args()
    if args.impl == "reference":
        return run_reference(args)
    if args.warmup < 3:
        args.warmup = 3

    import torch
    import torch.distributed as dist
    if not torch.cuda.is_available():
        raise SystemExit("bench.py needs a CUDA device: the product path has no CPU fallback")
    from paper_2411_18341_b200 import binding as phx

    world = int(os.environ.get("WORLD_SIZE", "1"))
    rank = int(os.environ.get("RANK", "0"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    torch.cuda.set_device(local)
    if world > 1:
        dist.init_process_group("nccl", device_id=torch.device("cuda", local))

    w = build_workload(args.workload)
    stream = torch.cuda.Stream()
    g = phx.grid_from_workload(w, variant=args.variant, stream=stream, device=f"cuda:{local}")
    for kv in filter(None, args.tune.split(",")):
        k, v = kv.split("=")
        g.set_tuning(k, int(v))
    variant = g.get_variant()

    def barrier():
        torch.cuda.synchronize()
        if world > 1:
            dist.barrier()
            torch.cuda.synchronize()

    # ---- device-resident throughput ---------------------------------------------------------------------
    def timed(steps):
        """CUDA events on the launching stream around `steps` RK4 steps, barrier + synchronize on both sides."""
        launches0 = g.get_launch_count()
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        barrier()
        e0.record(stream)
        g.step_rk4(steps)
        e1.record(stream)
        barrier()
        t_ms = max_over_ranks(e0.elapsed_time(e1), world)
        return t_ms, g.get_launch_count() - launches0

    g.step_rk4(args.warmup)
    barrier()
    sampler = ClockSampler(local)
    if rank == 0:
        sampler.start()
        time.sleep(0.25)
    t_wall0 = time.time()
    ms, launches = timed(args.steps)
    t_wall1 = time.time()
    clocks = sampler.stop(t_wall0, t_wall1) if rank == 0 else None
    cells = w.cells
    value = whole_job_value(world, cells, args.steps, ms)

    # the per-stage variant (the HBM-bound kernels of the north_star's >= 70 % target), timed the same way on a
    # shorter run, when the headline ran the fused step
    stage_info = None
    if variant != phx.PHX_VARIANT_STAGE and not args.no_stage_leg:
        g.select_variant(phx.PHX_VARIANT_STAGE)
        g.step_rk4(args.warmup)
        st_steps = max(8, args.steps // 4)
        st_ms, st_launches = timed(st_steps)
        st_bpc = algo_bytes_per_cell_step(w, phx.PHX_VARIANT_STAGE)
        st_val = whole_job_value(world, cells, st_steps, st_ms)
        st_gbs = st_bpc * cells * st_steps / (st_ms * 1e-3) / 1e9
        stage_info = {"variant": 1, "kernel": "phx::stage_kernel (4 launches per step)", "value": st_val, "unit": UNIT,
                      "steps": st_steps, "ms_per_step": st_ms / st_steps, "gpu_launches": int(st_launches),
                      "algorithmic_bytes_per_cell_step": st_bpc,
                      "roofline": {"bound": "hbm", "achieved": st_gbs, "unit": "GB/s"}}
        g.select_variant(variant)
    finite = bool(np.all(np.isfinite(g.read_field("psi_p")[0, :4])))

    # ---- end to end through the C ABI with host buffers ----------------------------------------------------
    # Every step uploads its state from pinned host memory, runs one RK4 step and downloads the result.  Two handles on two
    # streams alternate, so that the upload of one step overlaps the download of the previous one (PCIe is full duplex);
    # a handle is synchronised before its buffers are used again.
    stream2 = torch.cuda.Stream()
    g2 = phx.grid_from_workload(w, variant=args.variant, stream=stream2, device=f"cuda:{local}", upload=False)
    for kv in filter(None, args.tune.split(",")):
        k, v = kv.split("=")
        g2.set_tuning(k, int(v))
    handles = (g, g2)
    for gr in handles:
        gr.set_tuning("async_host_copies", 1)
    host_in = {k: torch.from_numpy(np.ascontiguousarray(v)).pin_memory() for k, v in w.fields.items()}
    host_out = [{k: torch.empty_like(v).pin_memory() for k, v in host_in.items()} for _ in handles]
    h2d = sum(v.numel() * v.element_size() for v in host_in.values())
    d2h = h2d

    def e2e_step(i):
        gr, out = handles[i % 2], host_out[i % 2]
        gr.sync()
        for k, v in host_in.items():
            gr.set_field(k, v)
        gr.step_rk4(1)
        for k, v in out.items():
            gr.read_field(k, v)
    for i in range(4):
        e2e_step(i)
    for gr in handles:
        gr.sync()
    barrier()
    t0 = time.perf_counter()
    for i in range(args.e2e_steps):
        e2e_step(i)
    for gr in handles:
        gr.sync()
    barrier()
    e2e_s = max_over_ranks(time.perf_counter() - t0, world)
    e2e_val = whole_job_value(world, cells, args.e2e_steps, e2e_s * 1e3)
    e2e_finite = bool(all(torch.isfinite(torch.view_as_real(v) if v.is_complex() else v).all() for o in host_out for v in o.values()))
    g2.destroy()

    if rank != 0:
        if world > 1:
            dist.destroy_process_group()
        return

    # ---- roofline of the dominant kernel ------------------------------------------------------------------------
    peak, peak_src = measured_peaks()
    bpc = algo_bytes_per_cell_step(w, variant, args.steps)
    kernels_per_step = launches / args.steps
    bytes_per_launch = bpc * cells / kernels_per_step
    launch_ms = ms / launches
    achieved = bytes_per_launch / (launch_ms * 1e-3) / 1e9
    comp = COMPULSORY_BYTES[w.model] * (2 if w.prec == "c64" else 1)
    kernel = {1: "phx::stage_kernel (4 launches per step)", 3: "phx::step_kernel (1 launch per step)",
              4: "phx::resident_kernel (1 launch for all steps)"}.get(variant, str(variant))
    hbm = {"achieved": achieved, "peak": peak, "unit": "GB/s", "frac": achieved / peak, "peak_source": peak_src,
           "algorithmic_bytes_per_cell_step": bpc, "bytes_per_launch": bytes_per_launch,
           "compulsory_bytes_per_cell_step": comp, "compulsory_frac": value / world * 1e9 * comp / 1e9 / peak}
    if variant in (phx.PHX_VARIANT_STEP, phx.PHX_VARIANT_RESIDENT):
        # the fused step moves the compulsory bytes only; it is bound by plain FP32/FP64 instruction issue
        fpc = algo_flops_per_cell_step(w)
        alu_peak = ALU_PEAK_TFLOPS[w.prec]
        tf = fpc * cells / kernels_per_step / (launch_ms * 1e-3) / 1e12
        roofline = {"bound": "alu", "achieved": tf, "peak": alu_peak, "unit": "TFLOP/s", "frac": tf / alu_peak,
                    "traffic": None, "peak_source": "derived: 148 SM x 128 (fp64: 64) lanes x 2 x 1.965 GHz, no tensor cores",
                    "kernel": kernel, "algorithmic_flops_per_cell_step": fpc, "flops_per_launch": fpc * cells / kernels_per_step,
                    "avg_launch_ms": launch_ms, "hbm": hbm}
    else:
        roofline = dict(hbm, bound="hbm", traffic=None, kernel=kernel, avg_launch_ms=launch_ms)
    if stage_info is not None:
        stage_info["roofline"].update(peak=peak, frac=stage_info["roofline"]["achieved"] / peak, peak_source=peak_src)
    # DRAM bytes per launch of this kernel from the committed `ncu --set full` capture (profiles/traffic.csv)
    traffic_file = os.path.join(ROOT, "profiles", "traffic.csv")
    if os.path.exists(traffic_file):
        try:
            for line in open(traffic_file):
                p = [x.strip() for x in line.split(",")]
                if len(p) >= 4 and p[0] == args.workload and p[1] == str(variant):
                    roofline["traffic"] = float(p[2])
                    roofline["traffic_source"] = p[3]
        except Exception:
            pass

    # ---- the oracle timed on this box's host cores (bounded sample) -----------------------------------------------
    cpu = None
    if not args.no_cpu_baseline and world == 1:
        ny = max(3, min(w.ny, (1 << 22) // w.nx))              # ~4M cells per step, ~0.4 s per step
        o = oracle_from_workload(w, ny)
        o.step_rk4(1)
        t0 = time.perf_counter()
        nst = 0
        while time.perf_counter() - t0 < 12.0:
            o.step_rk4(1)
            nst += 1
        dtc = time.perf_counter() - t0
        cpu = {"value": w.nx * ny * nst / dtc / 1e9, "unit": UNIT, "cores": 1, "kind": "oracle",
               "sample": f"{w.nx}x{ny} row slab of realisation 0, {nst} RK4 steps, fp64, single thread"}

    out = {
        "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps, "warmup": args.warmup,
        "ms_per_step": ms / args.steps, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
        "dtype": "f32" if w.prec == "c32" else "f64", "data": "synthetic",
        "config": {"workload": args.workload, "model": None, "grid": [w.nx, w.ny], "batch": w.batch, "precision": w.prec,
                   "variant": variant, "parallelism": "replicas only" if world > 1 else "single GPU",
                   "l2": f"working set {g.workspace.numel() / 2**20:.0f} MiB > 126 MB L2, no flush needed"
                   if g.workspace.numel() > 200e6 else "working set fits L2 (L2-resident regime, reported as such)",
                   "finite": finite},
        "clocks": clocks, "gpu_launches": int(launches),
        "e2e": {"value": e2e_val, "unit": UNIT, "h2d_bytes_per_step": h2d, "d2h_bytes_per_step": d2h,
                "rk4_steps_per_call": 1, "steps": args.e2e_steps, "finite": e2e_finite,
                "pipeline": "two handles on two streams: the upload of one step overlaps the download of the previous one"},
        "roofline": roofline, "cpu_baseline": cpu, "stage_variant": stage_info,
    }
    del out["config"]["model"]
    print(json.dumps(out))
    if world > 1:
        dist.destroy_process_group()


if __name__ == "__main__":
    main()
