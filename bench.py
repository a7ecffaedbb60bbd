#!/usr/bin/env python
"""bench.py — throughput of the hot path (BASELINE.json metric: cell-updates/s per RK3 step, fp64,
1 B200, and fraction of the fp64 roofline).

    python bench.py [--gpus N] [--steps K] [--warmup W] [--size n] [--dtype f64|f32] [--impl ours|reference]

A "step" is one pass of the whole hot path: jf_rk3_step = 3 x (halo fill, centre gradients, x/y/z
sweeps with WENO5 + HLLC + viscous flux, divergence, RK3 stage) on the Taylor-Green input of
BASELINE.json configs[4] (default 256^3 fp64: the size north_star's target is quoted at; the state is
719 MB, i.e. larger than the 126 MB L2, so every step streams from HBM — no L2 flush needed).
Prints ONE JSON line (rank 0).  N > 1: independent replicas, one per GPU (the path has no exchange
step on one GPU), barrier + max-over-ranks timing, value = all cells / time.
"""
import argparse
import json
import os
import subprocess
import sys
import threading
import time

ROOT = os.path.dirname(os.path.abspath(__file__))
sys.path.insert(0, ROOT)

METRIC = "cell-updates/s per RK3 step"
UNIT = "cell-updates/s"


def parse_args():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=20)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--size", type=int, default=256, help="n of the n^3 Taylor-Green box")
    ap.add_argument("--case", default="tgv", choices=["tgv", "channel"],
                    help="tgv: BASELINE.json configs[4] (default, the metric's workload); channel: configs[2] "
                         "(192x128x128, walls, Sutherland, body force, CFL time step taken every step)")
    ap.add_argument("--dtype", default="f64", choices=["f64", "f32", "f64t"],
                    help="f64t: the tangent solver (JF_F64_TANGENT: value + derivative w.r.t. the disturbance-wall parameters); "
                         "its roofline fields use the primal's flop count and fp64 peak (the tangent part is not counted)")
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--ref-size", type=int, default=96, help="n^3 sample the reference arm steps")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-e2e", action="store_true")
    ap.add_argument("--no-sweep", dest="sweep", action="store_false",
                    help="skip the other lines of configs[4] (384^3, 512^3 fp64, 512^3 fp32) the default run appends")
    ap.add_argument("--visc-order", type=int, default=4, choices=[4, 6],
                    help="order of the central dissipative-flux stencils: 4 (north_star, default) or 6 (PAPER.md:90, the "
                         "paper's DNS; with --case channel --dtype f32 this is the paper's own precision and dissipative scheme)")
    ap.add_argument("--decomp", default=None, metavar="Sx,Sy,Sz",
                    help="block-decomposition arm: one --size^3 block per rank, Sx*Sy*Sz ranks (PAPER.md:78-82)")
    return ap.parse_args()


# ---------------------------------------------------------------------------- flop model (oracle count)
def flop_model(n):
    """Algorithmic flops per interior cell from oracle/flop_model.json (written by
    oracle/count_flops.py from the oracle's counting build): step, one RHS, prim, grad."""
    with open(os.path.join(ROOT, "oracle", "flop_model.json")) as f:
        m = json.load(f)
    x = 1.0 / n
    ev = lambda key: sum(c * x ** k for k, c in enumerate(m[key][3]))
    return {k: ev(k) for k in ("step", "rhs", "prim", "grad")}


# ---------------------------------------------------------------------------- clocks
class ClockSampler:
    Q = ("index,clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,"
         "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,"
         "clocks_event_reasons.sw_power_cap")

    def __init__(self, index):
        self.index = index
        self.proc = None
        self.lines = []

    def start(self):
        try:
            self.proc = subprocess.Popen(["nvidia-smi", f"--query-gpu={self.Q}", "--format=csv,noheader,nounits",
                                          "-lms", "25", "-i", str(self.index)], stdout=subprocess.PIPE, text=True)
            self.t = threading.Thread(target=self._read, daemon=True)
            self.t.start()
        except OSError:
            self.proc = None

    def _read(self):
        for ln in self.proc.stdout:
            self.lines.append(ln.strip())

    def stop(self):
        if self.proc is None:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        self.proc.terminate()
        try:
            self.proc.wait(timeout=5)
        except subprocess.TimeoutExpired:
            self.proc.kill()
        sm, mx, pw, reasons = [], [], [], set()
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        for ln in self.lines:
            p = [s.strip() for s in ln.split(",")]
            if len(p) < 8:
                continue
            try:
                sm.append(float(p[1])); mx.append(float(p[2])); pw.append(float(p[3]))
            except ValueError:
                continue
            for nm, v in zip(names, p[4:8]):
                if v == "Active":
                    reasons.add(nm)
        sm.sort()
        return {"sm_mhz": sm[len(sm) // 2] if sm else None, "sm_max_mhz": max(mx) if mx else None,
                "power_w_max": max(pw) if pw else None, "samples": len(sm), "reasons": sorted(reasons)}


# ---------------------------------------------------------------------------- reference arm = the oracle
def oracle_throughput(n, steps, warmup, channel=False, visc_order=4):
    """The oracle as it stands (oracle/libora.so, -O2 -ffp-contract=off -fopenmp) on the host cores."""
    from oracle import ora
    from paper_2406_19494_b200 import cases
    case = cases.channel() if channel else cases.tgv(n)
    case.visc_order = visc_order
    o = ora.Oracle(case)
    U = o.state()

    def step():
        o.rk3_step(U, o.cfl_dt(U, case.cfl)[1] if channel else case.dt)

    for _ in range(warmup):
        step()
    t0 = time.perf_counter()
    for _ in range(steps):
        step()
    dt = time.perf_counter() - t0
    return case.cells * steps / dt, dt, os.cpu_count()


def run_reference(args):
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    val, secs, cores = oracle_throughput(args.ref_size, args.steps, args.warmup)
    sample = f"tgv {args.ref_size}^3 fp64, {args.steps} RK3 steps after {args.warmup} warm-up (same physics as the GPU arm's {args.size}^3 box)"
    line = {"impl": "reference", "metric": METRIC, "value": val, "unit": UNIT, "n_gpus": args.gpus, "steps": args.steps,
            "warmup": args.warmup, "ms_per_step": 1e3 * secs / args.steps, "higher_is_better": True,
            "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
            "config": {"workload": f"tgv{args.size} fp64 (BASELINE.json configs[4])", "reference": "CPU oracle (oracle/), host cores",
                       "sample": sample},
            "cpu_baseline": {"value": val, "unit": UNIT, "cores": cores, "kind": "oracle", "sample": sample},
            "e2e": {"value": val, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
            "gpu_launches": 0}
    print(json.dumps(line), flush=True)


# ---------------------------------------------------------------------------- multi-rank aggregation
def max_over_ranks(times_ms, world, device=None):
    """Replicas: every rank times its own box; the job's time is the slowest
    rank's.  Returns the element-wise MAX over ranks of the local millisecond timings."""
    if world <= 1:
        return [float(t) for t in times_ms]
    import torch
    import torch.distributed as dist
    t = torch.tensor([float(x) for x in times_ms], dtype=torch.float64, device=device)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return [float(x) for x in t]


def job_throughput(cells_per_rank, steps, world, ms):
    """Whole-job cell-updates/s: all ranks' cells x steps / the max-over-ranks time."""
    return world * cells_per_rank * steps / (ms * 1e-3)


# ---------------------------------------------------------------------------- our arm
def measured_peaks():
    ppath = os.path.join(ROOT, "MEASURED_PEAKS.json")
    return json.load(open(ppath)) if os.path.exists(ppath) else {}


def profile_row(kernel, n, dtype):
    """Row of profiles/traffic.csv (hand-copied from the committed ncu --set full capture; profiles/traffic.md
    names the command): DRAM bytes and executed FP64 thread-instructions per launch, averaged over the three
    stage launches of one step.  None for sizes / dtypes without a row."""
    tpath = os.path.join(ROOT, "profiles", "traffic.csv")
    if not os.path.exists(tpath):
        return None
    import csv
    with open(tpath) as f:
        for row in csv.DictReader(f):
            if row["kernel"] == kernel and int(row["size"]) == n and row["dtype"] == dtype:
                return row
    return None


def alu_peak(jf, dtype, local):
    """Measured ALU peak (jf_diag_alu_peak: register-resident FMA loop).  burst: best of three short launches;
    sustained: back to back for 1.5 s, median of the second half, with the SM clock sampled meanwhile."""
    burst, _ = jf.jf_diag_alu_peak(dtype, 4096)
    clk = ClockSampler(local)
    clk.start()
    samples, t_end = [], time.time() + 1.5
    while time.time() < t_end or len(samples) < 8:
        samples.append(jf.jf_diag_alu_peak(dtype, 4096)[0])
    c = clk.stop()
    tail = sorted(samples[len(samples) // 2:])
    return burst, tail[len(tail) // 2], c.get("sm_mhz")


def time_steps(torch, step, K, W, barrier, sampler=None):
    for _ in range(W):
        step()
    barrier()
    if sampler:
        sampler.start()
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    e0.record()
    for _ in range(K):
        step()
    e1.record()
    barrier()
    return e0.elapsed_time(e1)


def t_roof_ms(flops_cell_step, cells, dtype, peak_flops, hbm_gbs):
    """north_star: the slower of the path's FLOPs at the ALU peak and its algorithmic bytes at HBM bandwidth."""
    return max(flops_cell_step * cells / peak_flops, (320 if dtype == "f64" else 160) * cells / (hbm_gbs * 1e9)) * 1e3


def run_ours(args):
    import numpy as np
    import torch
    import torch.distributed as dist
    from paper_2406_19494_b200 import binding as jf, cases

    world = int(os.environ.get("WORLD_SIZE", "1"))
    rank = int(os.environ.get("RANK", "0"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device — libjf has no CPU fallback")
    torch.cuda.set_device(local)
    dev = torch.device("cuda", local)
    if world > 1:
        dist.init_process_group("nccl", device_id=dev)

    def barrier():
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    if args.decomp:
        return run_decomp(args, torch, dist, jf, cases, world, rank, local, dev, barrier)

    n, K, W = args.size, args.steps, max(args.warmup, 3)
    channel = args.case == "channel"
    case = cases.channel() if channel else cases.tgv(n)
    case.visc_order = args.visc_order
    solver = jf.Solver(case, args.dtype, device=str(dev))
    esz = {"f64": 8, "f32": 4, "f64t": 16}[args.dtype]
    U = solver.state()
    dt = case.dt
    state_bytes = U.numel() * esz

    def step(V=None):
        # fixed-dt configs (0, 4) time jf_rk3_step alone; CFL-driven configs (1-3) take the CFL reduction every step,
        # formed and consumed on the device (jf_cfl_dt_dev + jf_rk3_step_dev: no host round trip inside the loop)
        V = U if V is None else V
        if channel:
            solver.jf_cfl_dt_dev(V, case.cfl)
            solver.jf_rk3_step_dev(V)
        else:
            solver.jf_rk3_step(V, dt)

    # --- device-resident throughput: inputs in HBM, K steps between two events, nothing else on the stream
    clocks = ClockSampler(local)
    step()                                             # first call captures the step's CUDA graph
    l0 = solver.jf_launch_count()
    ms = time_steps(torch, step, K, W, barrier, clocks)
    launches = (solver.jf_launch_count() - l0) * K // (K + W)
    if channel and solver.jf_dev_time()[0] != 0:
        raise SystemExit("bench.py: device-side CFL reduction flagged an inadmissible state")
    # the same K steps once more with an event pair around every launch (jf_diag_timing; plain launches, no graph):
    # per-kernel durations for the roofline of the dominant kernel.  Kept out of the region above because the 30
    # extra event records per step cost 2 % at 256^3 and 10-40 % on the small boxes.
    solver.jf_diag_kernel_times()                      # reset
    solver.jf_diag_timing(True)
    ms_instr = time_steps(torch, step, K, 0, barrier)
    ktimes = solver.jf_diag_kernel_times()
    solver.jf_diag_timing(False)
    clk = clocks.stop()
    finite = solver.jf_cfl_dt(U, 1.0)[0] == 0          # the library's own reduction: every interior cell finite, rho, p > 0

    # --- end to end: host buffers, H2D of the input and D2H of the result inside every step.  Every step is one
    # independent job (its own input from pinned host memory, its own result back in pinned host memory); the jobs
    # are double-buffered on the device so that the upload of job i+1 and the download of job i-1 (two copy engines,
    # two side streams) overlap the kernels of job i on the solver's stream.
    e2e = None
    if not args.no_e2e:
        host_in = torch.empty(U.shape, dtype=U.dtype, pin_memory=True)
        host_in.copy_(solver.state().cpu() if args.dtype == "f64t" else torch.as_tensor(case.U0, dtype=U.dtype))
        # three device buffers: a buffer is busy for upload + kernels + download (13-16 + 7 + 13-16 ms at 256^3), so with two
        # of them a job takes half of that (19 ms: measured in round 1-2); with three the copies run back to back and the
        # PCIe link, both directions at once (measured: 15.7 ms for 719 MB each way), is the limit
        NBUF = 3
        host_out = [torch.empty(U.shape, dtype=U.dtype, pin_memory=True) for _ in range(NBUF)]
        bufs = [U] + [torch.empty_like(U) for _ in range(NBUF - 1)]
        cur = torch.cuda.current_stream(dev)
        s_in, s_out = torch.cuda.Stream(dev), torch.cuda.Stream(dev)

        def pipeline(njobs):
            d2h_done = [None] * NBUF
            for i in range(njobs):
                b = i % NBUF
                with torch.cuda.stream(s_in):
                    if d2h_done[b] is not None:
                        s_in.wait_event(d2h_done[b])           # the buffer's previous result has left the device
                    bufs[b].copy_(host_in, non_blocking=True)
                    ev_in = torch.cuda.Event(); ev_in.record(s_in)
                cur.wait_event(ev_in)
                step(bufs[b])
                ev_c = torch.cuda.Event(); ev_c.record(cur)
                with torch.cuda.stream(s_out):
                    s_out.wait_event(ev_c)
                    host_out[b].copy_(bufs[b], non_blocking=True)
                    d2h_done[b] = torch.cuda.Event(); d2h_done[b].record(s_out)
            for ev in d2h_done:
                if ev is not None:
                    cur.wait_event(ev)

        Ke = K
        pipeline(NBUF)
        barrier()
        t0 = torch.cuda.Event(enable_timing=True); t1 = torch.cuda.Event(enable_timing=True)
        t0.record()
        pipeline(Ke)
        t1.record()
        barrier()
        ms_e2e = t0.elapsed_time(t1)
        e2e = (ms_e2e, Ke)
        e2e_finite = bool(torch.isfinite(host_out[(Ke - 1) % NBUF]).all().item())

    # --- the other lines of configs[4] (N = 1, default workload only): 384^3 and 512^3 fp64, 512^3 fp32
    sweep = None
    if world == 1 and not channel and args.sweep and n == 256 and args.dtype == "f64":
        del solver, U
        if e2e:
            del bufs, host_in, host_out
        torch.cuda.empty_cache()
        sweep = []
        for sn, sdt in ((384, "f64"), (512, "f64"), (512, "f32")):
            sc = cases.tgv(sn)
            ss = jf.Solver(sc, sdt, device=str(dev))
            SU = ss.state()
            sck = ClockSampler(local)
            ss.jf_rk3_step(SU, sc.dt)
            sms = time_steps(torch, lambda: ss.jf_rk3_step(SU, sc.dt), 5, 3, barrier, sck)
            sclk = sck.stop()
            sweep.append({"size": sn, "dtype": sdt, "cells": sc.cells, "steps": 5, "ms_per_step": sms / 5,
                          "value": sc.cells * 5 / (sms * 1e-3), "sm_mhz": sclk.get("sm_mhz"), "reasons": sclk.get("reasons"),
                          "finite": ss.jf_cfl_dt(SU, 1.0)[0] == 0})
            del ss, SU
            torch.cuda.empty_cache()

    # --- max over ranks
    if world > 1:
        ms, e2e_ms = max_over_ranks([ms, e2e[0] if e2e else 0.0], world, dev)
        e2e = (e2e_ms, e2e[1]) if e2e else None
    if rank != 0:
        if world > 1:
            dist.destroy_process_group()
        return

    cells = case.cells
    value = job_throughput(cells, K, world, ms)
    fm = flop_model(n)
    if channel:                                        # one step of config 2, counted by the oracle at full size
        with open(os.path.join(ROOT, "oracle", "flop_model.json")) as f:
            ch = json.load(f)["channel_step_order6" if args.visc_order == 6 else "channel_step"][3]
        fm = {k: v * ch / fm["step"] for k, v in fm.items()}   # pieces scaled like the Taylor-Green split
    # roofline of the dominant kernel (bound: plain FP64/FP32 ALUs; nothing here is a contraction).  The step kernels
    # are timed inside a long run, so the sustained peak is the roofline's; the burst figure is reported beside it.
    # The peak loop holds the maximum SM clock while the step runs into the board's power cap, so the fraction at the
    # clock the step actually ran at is reported too (peak scaled by run clock / peak-loop clock).
    pdt = "f32" if args.dtype == "f32" else "f64"
    peak_burst, peak_flops, peak_mhz = alu_peak(jf, pdt, local)
    run_mhz = clk.get("sm_mhz")
    clock_ratio = (run_mhz / peak_mhz) if (run_mhz and peak_mhz) else None
    sweep_flops = (fm["rhs"] - fm["prim"] - fm["grad"]) / 3.0           # one direction: WENO5+HLLC+viscous face+divergence
    rk_flops = (fm["step"] - 3.0 * fm["rhs"]) / 3.0                    # stage update
    alg = {"sweep_x_kernel": sweep_flops + fm["prim"] / 3.0, "sweep_yz_kernel<y>": sweep_flops + fm["prim"] / 3.0,
           "sweep_yz_kernel<z>+rk": sweep_flops + fm["prim"] / 3.0 + rk_flops, "gradient_kernel": fm["grad"]}
    dom = max((k for k in ktimes if ktimes[k][1] > 0), key=lambda k: ktimes[k][0])
    dom_ms, dom_n = ktimes[dom]
    dom_flops = alg.get(dom, 0.0) * cells
    dom_s = dom_ms / dom_n * 1e-3 if dom_n else None
    achieved = dom_flops / dom_s / 1e12 if dom_n else 0.0
    # measured DRAM bytes and executed FP64 instructions of the dominant kernel (committed ncu capture)
    row = None if channel else profile_row(dom, n, args.dtype)
    bdt = "f32" if args.dtype == "f32" else "f64"       # bytes / flops model of the value part
    traffic = float(row["dram_bytes_per_launch"]) if row else None
    executed = None
    if row and row.get("dfma_thread_inst"):
        ex_flops = 2.0 * float(row["dfma_thread_inst"]) + float(row["dadd_thread_inst"]) + float(row["dmul_thread_inst"])
        executed = {"flops_per_launch": ex_flops, "achieved": ex_flops / dom_s / 1e12, "frac": ex_flops / dom_s / peak_flops,
                    "numerator": "2*DFMA + DADD + DMUL thread-instructions of the launch (ncu smsp__sass_thread_inst_executed_op_*; "
                                 "divisions / square roots appear as the Newton steps they are executed as)"}
    peaks = measured_peaks()
    hbm = peaks.get("hbm_gbs", 6650.0)
    troof = t_roof_ms(fm["step"], cells, bdt, peak_flops, hbm)
    if sweep:
        for ln in sweep:
            sfm = flop_model(ln["size"])
            pk = peak_flops if ln["dtype"] == args.dtype else alu_peak(jf, ln["dtype"], local)[1]
            tr = t_roof_ms(sfm["step"], ln["cells"], ln["dtype"], pk, hbm)
            ln["roofline_step_frac"] = tr / ln["ms_per_step"]
            ln["roofline_step_frac_at_run_clock"] = (tr / ln["ms_per_step"] * peak_mhz / ln["sm_mhz"]) if (peak_mhz and ln.get("sm_mhz")) else None
            ln["peak_tflops"] = pk / 1e12
    line = {
        "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": K, "warmup": W,
        "ms_per_step": ms / K, "ms_per_step_with_per_launch_events": ms_instr / K,
        "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
        "dtype": args.dtype, "data": "synthetic",
        "config": {"workload": ("channel 192x128x128 (BASELINE.json configs[2]: isothermal walls, Sutherland, body force, tanh y grid; "
                                "jf_cfl_dt_dev + jf_rk3_step_dev every step)" + (", sixth-order central dissipative flux" if args.visc_order == 6 else "")) if channel else
                               f"tgv{n} {dict(f64='fp64', f32='fp32', f64t='fp64 tangent solver')[args.dtype]} (BASELINE.json configs[4]: Taylor-Green {n}^3, dt=1e-3)"
                               + (" [sixth-order dissipative flux; flops counted for the fourth-order scheme]" if args.visc_order == 6 else ""),
                   "cells": cells, "state_bytes": state_bytes, "l2": "inputs larger than L2 (no flush)" if state_bytes > 126e6 else "state fits L2",
                   "parallelism": f"replicas x{world}" if world > 1 else "1 GPU", "finite": finite,
                   "launch": "CUDA graph of the 15 kernels of a step, replayed (+ 1 one-thread kernel carrying a host dt)"},
        "clocks": clk,
        "gpu_launches": int(launches),
        "roofline": {"bound": "alu", "kernel": dom, "achieved": achieved, "peak": peak_flops / 1e12, "unit": "TFLOP/s",
                     "frac": achieved / (peak_flops / 1e12), "traffic": traffic,
                     "numerator": "algorithmic flops: the oracle's own operation count (add/sub/mul/min/max/div/sqrt = 1), oracle/flop_model.json",
                     "frac_at_run_clock": achieved / (peak_flops / 1e12) / clock_ratio if clock_ratio else None,
                     "peak_loop_sm_mhz": peak_mhz, "run_sm_mhz": run_mhz,
                     "executed": executed,
                     "peak_burst": peak_burst / 1e12, "frac_of_burst": achieved / (peak_burst / 1e12),
                     "peak_source": "measured live, sustained: jf_diag_alu_peak register-resident FMA loop back to back for 1.5 s (DESIGN.md)",
                     "flops_per_cell_launch": alg.get(dom), "avg_launch_ms": dom_ms / dom_n if dom_n else None},
        "roofline_step": {"flops_per_cell_step": fm["step"], "t_roof_ms": troof, "frac": troof / (ms / K),
                          "frac_at_run_clock": troof / (ms / K) / clock_ratio if clock_ratio else None,
                          "frac_of_burst_peak": t_roof_ms(fm["step"], cells, bdt, peak_burst, hbm) / (ms / K),
                          "hbm_gbs": hbm, "hbm_source": "measured" if peaks else "fallback"},
        "kernels_ms_per_step": {k: v[0] / K for k, v in ktimes.items() if v[1]},
    }
    if sweep:
        line["sweep"] = sweep
    if e2e:
        line["e2e"] = {"value": job_throughput(cells, e2e[1], world, e2e[0]), "unit": UNIT,
                       "h2d_bytes_per_step": state_bytes, "d2h_bytes_per_step": state_bytes, "ms_per_step": e2e[0] / e2e[1],
                       "pipeline": "three device buffers: H2D of job i+1 and D2H of job i-1 overlap the kernels of job i; bound by the PCIe link (both directions at once)", "finite": e2e_finite}
    if world == 1 and not args.no_cpu_baseline:
        # bounded sample: one RK3 step of the SAME input on the host cores (the oracle as it stands)
        nb = min(n, 256)
        val, secs, cores = oracle_throughput(nb, 1, 0, channel, args.visc_order)
        line["cpu_baseline"] = {"value": val, "unit": UNIT, "cores": cores, "kind": "oracle",
                                "sample": (f"1 step (cfl_dt + RK3) of the channel 192x128x128 fp64 ({secs:.1f} s)" if channel
                                           else f"1 RK3 step of tgv{nb} fp64 ({secs:.1f} s)")}
    print(json.dumps(line), flush=True)
    if world > 1:
        dist.destroy_process_group()


# ---------------------------------------------------------------------------- block decomposition arm
def pid_seconds(ms_per_step, ranks, dof):
    """The paper's performance index, Eq. 9: PID = wall time per step x #ranks / #DOF."""
    return ms_per_step * 1e-3 * ranks / dof


def run_decomp(args, torch, dist, jf, cases, world, rank, local, dev, barrier):
    """--decomp Sx,Sy,Sz: the paper's own parallel strategy, one n^3 Taylor-Green block per rank
    (weak scaling), halos of inter-block faces exchanged point-to-point three times per RK stage (decomp.RankBlock).
    Needs Sx*Sy*Sz ranks.  Prints cell-updates/s of the whole job and the PID of Eq. 9 next to it."""
    from paper_2406_19494_b200 import decomp
    S = tuple(int(v) for v in args.decomp.split(","))
    if len(S) != 3 or S[0] * S[1] * S[2] != world:
        raise SystemExit(f"bench.py --decomp {args.decomp}: needs {S[0] * S[1] * S[2] if len(S) == 3 else '?'} ranks, have {world}")
    n, K, W = args.size, args.steps, max(args.warmup, 3)
    if world == 1 and not dist.is_initialized():       # a single block: the arm still goes through RankBlock (no exchange faces)
        os.environ.setdefault("MASTER_ADDR", "127.0.0.1")
        os.environ.setdefault("MASTER_PORT", "29533")
        dist.init_process_group("nccl", rank=0, world_size=1, device_id=dev)
    part = decomp.tgv_part(n, S, rank)
    rb = decomp.RankBlock(None, S, args.dtype, device=str(dev), part=part)
    dt = part.case.dt
    clocks = ClockSampler(local)
    ms = time_steps(torch, lambda: rb.jf_rk3_step(dt), K, W, barrier, clocks)
    clk = clocks.stop()
    finite = rb.jf_cfl_dt(1.0)[0] == 0
    (ms,) = max_over_ranks([ms], world, dev)
    if rank == 0:
        cells = part.case.cells
        line = {"metric": METRIC, "value": job_throughput(cells, K, world, ms), "unit": UNIT, "n_gpus": world, "steps": K,
                "warmup": W, "ms_per_step": ms / K, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
                "dtype": args.dtype, "data": "synthetic",
                "config": {"workload": f"tgv {n}^3 per rank, blocks {S[0]}x{S[1]}x{S[2]} (PAPER.md:78-82 decomposition; global "
                                       f"{n * S[0]}x{n * S[1]}x{n * S[2]})", "cells_per_rank": cells, "finite": finite,
                           "parallelism": f"domain decomposition {S[0]}x{S[1]}x{S[2]}, halo exchange by NCCL point-to-point",
                           "exchange_bytes_per_rank_per_step": rb.exchange_bytes_per_step()},
                "clocks": clk, "gpu_launches": int(rb.solver.jf_launch_count() * K // (K + W)),
                "pid": {"eq": "PAPER.md:130 Eq. 9: wall time per step x ranks / DOF",
                        "dof_cells": pid_seconds(ms / K, world, cells * world),
                        "dof_cells_x5": pid_seconds(ms / K, world, 5 * cells * world), "unit": "s"}}
        print(json.dumps(line), flush=True)
    if dist.is_initialized():
        dist.destroy_process_group()


if __name__ == "__main__":
    a = parse_args()
    if a.impl == "reference":
        run_reference(a)
    else:
        run_ours(a)
