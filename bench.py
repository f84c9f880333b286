#!/usr/bin/env python
"""bench.py -- throughput of the RK4 hot path on B200 (BASELINE.json metric: grid-cell RK4 steps per second).

    python bench.py [--gpus N] [--steps K] [--warmup W] [--workload NAME] [--variant V] [--impl reference]

A "step" is one RK4 step (all four stages, plus noise where the workload has it) over the whole grid /
ensemble.  `value` times blocks of exactly K steps with the state resident in HBM (CUDA events on the launching
stream, barrier + synchronize on both sides, max over ranks): the block is repeated until the timed region is at
least 0.5 s long (at least 5 blocks) and the MEDIAN block is reported, so that a short
--steps does not turn the measurement into a millisecond sample.  `e2e` times the same metric through the C ABI with
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


def build_workload(name, quick=False):
    """quick=True (the short other_workloads timings): the 16384^2 spinor fields are a 2048^2 recipe tile repeated 8 x 8."""
    from paper_2411_18341_b200 import workloads as wl
    if quick and name == "cfg4_16384_c32":
        return wl.cfg4(16384, "c32", tile=2048)
    table = {
        "cfg1": lambda: wl.cfg1(),
        "cfg2_1024_c32": lambda: wl.cfg2(1024, "c32"), "cfg2_1024_c64": lambda: wl.cfg2(1024, "c64"),
        "cfg2_4096_c32": lambda: wl.cfg2(4096, "c32"), "cfg2_4096_c64": lambda: wl.cfg2(4096, "c64"),
        # beyond BASELINE's sizes (the scalar model on larger grids: the fused step's rate away from single-wave effects)
        "cfg2_8192_c32": lambda: wl.cfg2(8192, "c32", tile=2048), "cfg2_16384_c32": lambda: wl.cfg2(16384, "c32", tile=2048),
        "cfg3_4096_c32": lambda: wl.cfg3(4096, "c32"),
        "cfg4_16384_c32": lambda: wl.cfg4(16384, "c32"), "cfg4_8192_c32": lambda: wl.cfg4(8192, "c32"),
        "cfg5_512x256_c32": lambda: wl.cfg5(256, 512, "c32"),
        # spinor with reservoirs (the paper's full 24-buffer system, Example 3) at its 500^2 and at a 4096^2 shape
        "ex3_500_c32": lambda: wl.example3(500, "c32"), "ex3_4096_c32": lambda: wl.example3(4096, "c32"),
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


# SURVEY.md section 8(d)'s own flop count per cell-step (scalar 130, reservoir + 50, spinor 2 x 170), next to DESIGN.md's.
SURVEY_FLOPS = {"scalar": 130, "reservoir": 180, "spinor": 340, "spinor_reservoir": 440}


def read_traffic():
    """profiles/traffic.csv: (workload, variant) -> (DRAM bytes per launch from the ncu capture, source)."""
    out = {}
    path = os.path.join(ROOT, "profiles", "traffic.csv")
    if os.path.exists(path):
        for line in open(path):
            p = [x.strip() for x in line.split(",", 3)]
            try:
                out[(p[0], int(p[1]))] = (float(p[2]), p[3])
            except (ValueError, IndexError):
                continue
    return out


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


def oracle_from_workload(w, ny=None, openmp=False):
    """The oracle as it stands on (a row-slab sample of) the workload.  openmp=True: the same source built with its
    OpenMP pragmas honoured (all host cores; the parity oracle is the single-threaded build)."""
    import oracle as orc
    orc.select_build(openmp)
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
    ap.add_argument("--min-seconds", type=float, default=0.5, help="floor of the timed region (blocks of --steps steps)")
    ap.add_argument("--no-other-workloads", action="store_true", help="skip the short timings of the other BASELINE configs")
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
    def timed(gr, steps):
        """CUDA events on the launching stream around `steps` RK4 steps, barrier + synchronize on both sides."""
        launches0 = gr.get_launch_count()
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        barrier()
        e0.record(stream)
        gr.step_rk4(steps)
        e1.record(stream)
        barrier()
        t_ms = max_over_ranks(e0.elapsed_time(e1), world)
        return t_ms, gr.get_launch_count() - launches0

    def timed_blocks(gr, steps, min_seconds, min_blocks=5, max_blocks=4000):
        """Blocks of exactly `steps` steps back to back on the stream, each bracketed by CUDA events, the whole region by
        barrier + synchronize; returns (median block ms (max over ranks), launches in the region, blocks, region ms)."""
        t1, _ = timed(gr, steps)                               # sizes the region (and is one more warm-up)
        nb = int(min(max_blocks, max(min_blocks, np.ceil(min_seconds * 1e3 / max(t1, 1e-3)))))
        if world > 1:                                          # every rank runs the same number of blocks
            nb = int(max_over_ranks(nb, world))
        launches0 = gr.get_launch_count()
        ev = [torch.cuda.Event(enable_timing=True) for _ in range(nb + 1)]
        barrier()
        ev[0].record(stream)
        for b in range(nb):
            gr.step_rk4(steps)
            ev[b + 1].record(stream)
        barrier()
        blocks_ms = [ev[b].elapsed_time(ev[b + 1]) for b in range(nb)]
        med = max_over_ranks(statistics.median(blocks_ms), world)
        return med, gr.get_launch_count() - launches0, nb, max_over_ranks(ev[0].elapsed_time(ev[nb]), world)

    g.step_rk4(args.warmup)
    barrier()
    sampler = ClockSampler(local)
    if rank == 0:
        sampler.start()
        time.sleep(0.25)
    t_wall0 = time.time()
    ms, launches, n_blocks, region_ms = timed_blocks(g, args.steps, args.min_seconds)
    t_wall1 = time.time()
    clocks = sampler.stop(t_wall0, t_wall1) if rank == 0 else None
    cells = w.cells
    value = whole_job_value(world, cells, args.steps, ms)
    launches_per_block = launches / n_blocks

    # the per-stage variant (the HBM-bound kernels of the north_star's >= 70 % target), timed the same way on a
    # shorter run, when the headline ran the fused step
    stage_info = None
    if variant != phx.PHX_VARIANT_STAGE and not args.no_stage_leg:
        g.select_variant(phx.PHX_VARIANT_STAGE)
        g.step_rk4(args.warmup)
        st_steps = max(8, args.steps // 4)
        st_ms, st_launches, st_blocks, _ = timed_blocks(g, st_steps, args.min_seconds / 2)
        st_launches //= st_blocks
        st_bpc = algo_bytes_per_cell_step(w, phx.PHX_VARIANT_STAGE)
        st_val = whole_job_value(world, cells, st_steps, st_ms)
        st_gbs = st_bpc * cells * st_steps / (st_ms * 1e-3) / 1e9
        stage_info = {"variant": 1, "kernel": "phx::stage_kernel (4 launches per step)", "value": st_val, "unit": UNIT,
                      "steps": st_steps, "ms_per_step": st_ms / st_steps, "gpu_launches": int(st_launches),
                      "algorithmic_bytes_per_cell_step": st_bpc,
                      "roofline": {"bound": "hbm", "achieved": st_gbs, "unit": "GB/s"}}
        g.select_variant(variant)
    finite = bool(np.all(np.isfinite(g.read_field("psi_p")[0, :4])))
    ws_bytes = g.workspace.numel()

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
    # Primary: the HBM roof (the lower roof of the model: 130-160 flop per 20 B is below the machine balance of 11 flop/B)
    # with the ALGORITHMIC bytes of the kernel that ran: achieved = bytes per launch / average launch duration.
    peak, peak_src = measured_peaks()
    bpc = algo_bytes_per_cell_step(w, variant, args.steps)
    kernels_per_step = launches_per_block / args.steps
    bytes_per_launch = bpc * cells / kernels_per_step
    launch_ms = ms / launches_per_block
    achieved = bytes_per_launch / (launch_ms * 1e-3) / 1e9
    comp = COMPULSORY_BYTES[w.model] * (2 if w.prec == "c64" else 1)
    kernel = {1: "phx::stage_kernel (4 launches per step)", 3: "phx::step_kernel (1 launch per step)",
              4: "phx::resident_kernel (1 launch for all steps)"}.get(variant, str(variant))
    roofline = {"bound": "hbm", "achieved": achieved, "peak": peak, "unit": "GB/s", "frac": achieved / peak, "traffic": None,
                "peak_source": peak_src, "kernel": kernel, "avg_launch_ms": launch_ms,
                "algorithmic_bytes_per_cell_step": bpc, "bytes_per_launch": bytes_per_launch,
                "compulsory_bytes_per_cell_step": comp, "compulsory_frac": value / world * 1e9 * comp / 1e9 / peak}
    if variant in (phx.PHX_VARIANT_STEP, phx.PHX_VARIANT_RESIDENT):
        # what actually limits the fused kernels is FP32/FP64 instruction issue: the same run against the
        # plain-ALU peak, nested; flops as SURVEY.md 8(d) counts them (130 per scalar cell-step) and as DESIGN.md counts them
        fpc = algo_flops_per_cell_step(w)
        alu_peak = ALU_PEAK_TFLOPS[w.prec]
        tf = fpc * cells / kernels_per_step / (launch_ms * 1e-3) / 1e12
        roofline["alu"] = {"achieved": tf, "peak": alu_peak, "unit": "TFLOP/s", "frac": tf / alu_peak,
                           "peak_source": "derived: 148 SM x 128 (fp64: 64) lanes x 2 x 1.965 GHz, no tensor cores",
                           "algorithmic_flops_per_cell_step": fpc,
                           "frac_with_survey_flop_count": tf / alu_peak * SURVEY_FLOPS.get(w.model, fpc) / fpc}
    # DRAM bytes per launch of this kernel from the committed `ncu --set full` captures (profiles/traffic.csv)
    traffic = read_traffic()
    if (args.workload, variant) in traffic:
        roofline["traffic"], roofline["traffic_source"] = traffic[(args.workload, variant)]
        roofline["frac_ncu_bytes"] = roofline["traffic"] / (launch_ms * 1e-3) / 1e9 / peak
    hbm_target = None
    if stage_info is not None:
        r = stage_info["roofline"]
        r.update(peak=peak, frac=r["achieved"] / peak, peak_source=peak_src)
        if (args.workload, 1) in traffic:
            tb, src = traffic[(args.workload, 1)]
            r["traffic"], r["traffic_source"] = tb, src
            r["frac_ncu_bytes"] = tb / (stage_info["ms_per_step"] / 4 * 1e-3) / 1e9 / peak
        # the north_star target (>= 70 % of the HBM roofline, bytes per cell-step from the ncu counters) is written for the
        # per-stage kernels; the fused step moves 6.4x fewer bytes and is judged by compulsory_frac / the ALU fraction
        f_ncu = r.get("frac_ncu_bytes")
        hbm_target = {"variant": 1, "frac_algorithmic_bytes": r["frac"], "frac_ncu_bytes": f_ncu,
                      "met": bool((f_ncu if f_ncu is not None else r["frac"]) >= 0.70)}

    # ---- short timings of the other BASELINE configs (STEP / AUTO and STAGE), so that every size the north_star names is
    # driver-visible: cfg4 16384^2, cfg3, cfg5, cfg2 fp64 (about 0.2 s of GPU time each) -------------------------------------
    others = None
    if not args.no_other_workloads and world == 1 and args.workload == "cfg2_4096_c32":
        others = {}
        g.destroy()
        del g
        torch.cuda.empty_cache()
        for name in ("cfg2_4096_c64", "cfg3_4096_c32", "cfg5_512x256_c32", "cfg4_16384_c32", "cfg2_1024_c32", "cfg2_16384_c32"):
            ow = build_workload(name, quick=True)
            og = phx.grid_from_workload(ow, stream=stream, device=f"cuda:{local}")
            rec = {}
            for vname, v in (("auto", phx.PHX_VARIANT_AUTO), ("stage", phx.PHX_VARIANT_STAGE))[:1 if name == "cfg2_16384_c32" else 2]:
                og.select_variant(v)
                vv = og.get_variant()
                og.step_rk4(5)
                o_steps = 16 if "16384" in name else 64
                o_ms, o_l, o_nb, _ = timed_blocks(og, o_steps, 0.2)
                val = ow.cells * o_steps / (o_ms * 1e-3) / 1e9
                ob = algo_bytes_per_cell_step(ow, vv, o_steps)
                oc = COMPULSORY_BYTES[ow.model] * (2 if ow.prec == "c64" else 1)
                rec[vname] = {"variant": vv, "value": val, "unit": UNIT, "ms_per_step": o_ms / o_steps, "steps": o_steps,
                              "blocks": o_nb, "algorithmic_bytes_per_cell_step": ob, "hbm_frac": val * ob / peak,
                              "compulsory_frac": val * oc / peak}
                if (name, vv) in traffic:
                    kps = o_l / o_nb / o_steps
                    rec[vname]["hbm_frac_ncu_bytes"] = traffic[(name, vv)][0] * kps / (o_ms / o_steps * 1e-3) / 1e9 / peak
            rec["finite"] = bool(np.all(np.isfinite(og.read_field("psi_p")[0, :2])))
            others[name] = rec
            og.destroy()
            del og, ow
            torch.cuda.empty_cache()

    # ---- the oracle timed on this box's host cores (bounded samples): as it stands on one core, and the same source with
    # its OpenMP pragmas honoured on all cores ----------------------------------------------------------
    cpu = None
    if not args.no_cpu_baseline and world == 1:
        ny = max(3, min(w.ny, (1 << 22) // w.nx))              # ~4M cells per step, ~0.4 s per step

        def time_oracle(openmp, budget):
            o = oracle_from_workload(w, ny, openmp=openmp)
            o.step_rk4(1)
            t0 = time.perf_counter()
            nst = 0
            while time.perf_counter() - t0 < budget:
                o.step_rk4(1)
                nst += 1
            return w.nx * ny * nst / (time.perf_counter() - t0) / 1e9, nst
        v1, n1 = time_oracle(False, 10.0)
        ncores = len(os.sched_getaffinity(0))
        os.environ.setdefault("OMP_NUM_THREADS", str(ncores))
        vn, nn_ = time_oracle(True, 8.0)
        import oracle as orc
        orc.select_build(False)
        cpu = {"value": v1, "unit": UNIT, "cores": 1, "kind": "oracle",
               "sample": f"{w.nx}x{ny} row slab of realisation 0, {n1} RK4 steps, fp64, single thread",
               "all_cores": {"value": vn, "unit": UNIT, "cores": ncores, "kind": "oracle, OpenMP over the rows of each full-grid loop",
                             "sample": f"{w.nx}x{ny} row slab, {nn_} RK4 steps"}}

    out = {
        "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps, "warmup": args.warmup,
        "ms_per_step": ms / args.steps, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
        "dtype": "f32" if w.prec == "c32" else "f64", "data": "synthetic",
        "config": {"workload": args.workload, "model": None, "grid": [w.nx, w.ny], "batch": w.batch, "precision": w.prec,
                   "variant": variant, "parallelism": "replicas only" if world > 1 else "single GPU",
                   "l2": f"working set {ws_bytes / 2**20:.0f} MiB > 126 MB L2, no flush needed"
                   if ws_bytes > 200e6 else "working set fits L2 (L2-resident regime, reported as such)",
                   "finite": finite},
        "timed_blocks": n_blocks, "timed_region_ms": region_ms, "block": "median of the blocks of `steps` steps",
        "clocks": clocks, "gpu_launches": int(launches), "gpu_launches_per_block": launches_per_block,
        "e2e": {"value": e2e_val, "unit": UNIT, "h2d_bytes_per_step": h2d, "d2h_bytes_per_step": d2h,
                "rk4_steps_per_call": 1, "steps": args.e2e_steps, "finite": e2e_finite,
                "pipeline": "two handles on two streams: the upload of one step overlaps the download of the previous one"},
        "roofline": roofline, "cpu_baseline": cpu, "stage_variant": stage_info, "hbm_target": hbm_target,
        "other_workloads": others,
    }
    del out["config"]["model"]
    print(json.dumps(out))
    if world > 1:
        dist.destroy_process_group()


if __name__ == "__main__":
    main()
