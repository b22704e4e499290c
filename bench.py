#!/usr/bin/env python
"""bench.py -- one JSON line with the headline metric of BASELINE.json:
band*dir*cell updates/s per sweep (whole source iterations: sweep + moments + dT/q/residual update).

  python bench.py [--gpus N] [--steps K] [--warmup W] [--config 4] [--impl ours|reference]

A "step" is one source iteration of the whole hot path on one seeded
synthetic problem (workloads.config(k)).  N > 1 (torchrun): replicas only -- every rank runs an
independent copy of the problem, value = sum of updates / max-over-ranks time.
`--impl reference` times the CPU oracle as it stands on the host cores (rank 0 only).
"""
import argparse
import json
import os
import subprocess
import sys
import threading
import time

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

METRIC = "band*dir*cell updates/s per sweep"
UNIT = "updates/s"
FLOP_PER_UPDATE = 16.0        # 3 FMA + 1 MUL (recurrence) + 4 FMA (moments), SURVEY.md 8(a)/DESIGN.md
SM_COUNT, SM_MAX_HZ = 148, 1.965e9
# plain-ALU peaks derived from unit counts x max clock: FP32 128 FMA/clk/SM,
# FP64 64 FMA/clk/SM
PEAK_TFLOPS = {"f32": SM_COUNT * 128 * 2 * SM_MAX_HZ / 1e12, "f64": SM_COUNT * 64 * 2 * SM_MAX_HZ / 1e12}
# algorithmic HBM bytes per sweep (cell fields + boundary store read and written once)
ALGORITHMIC_BYTES = {1: 11.2e6, 2: 17.7e6, 3: 63.6e6, 4: 964e6}


def parse():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=20)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--config", type=int, default=4, help="BASELINE.json configs[k]")
    ap.add_argument("--precision", choices=["config", "f64", "f32"], default="config")
    ap.add_argument("--impl", choices=["ours", "reference"], default="ours")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-converge", action="store_true", help="skip the time-to-eps_T<=1e-8 run (part of the metric)")
    ap.add_argument("--converge", action="store_true", help="(default; kept for compatibility)")
    return ap.parse_args()


class ClockSampler:
    """nvidia-smi clocks / throttle reasons sampled every 200 ms during the timed region."""
    Q = ("clocks.sm,clocks.max.sm,clocks_event_reasons.hw_slowdown,clocks_event_reasons.hw_thermal_slowdown,"
         "clocks_event_reasons.sw_thermal_slowdown,clocks_event_reasons.sw_power_cap")

    def __init__(self, index):
        self.rows, self.proc, self.index = [], None, index

    def start(self):
        try:
            self.proc = subprocess.Popen(["nvidia-smi", "-i", str(self.index), f"--query-gpu={self.Q}",
                                          "--format=csv,noheader,nounits", "-lms", "200"],
                                         stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
            self.t = threading.Thread(target=self._read, daemon=True)
            self.t.start()
        except OSError:
            self.proc = None

    def _read(self):
        for line in self.proc.stdout:
            self.rows.append([x.strip() for x in line.split(",")])

    def stop(self):
        if not self.proc:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        time.sleep(0.25)
        self.proc.terminate()
        self.t.join(timeout=2)
        sm = sorted(int(r[0]) for r in self.rows if r and r[0].isdigit())
        mx = [int(r[1]) for r in self.rows if len(r) > 1 and r[1].isdigit()]
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        reasons = [n for k, n in enumerate(names) if any(len(r) > 2 + k and r[2 + k] == "Active" for r in self.rows)]
        return {"sm_mhz": sm[len(sm) // 2] if sm else None, "sm_max_mhz": max(mx) if mx else None,
                "reasons": reasons, "samples": len(sm)}


def ncu_traffic(k, dtype):
    """dram__bytes_read.sum + dram__bytes_write.sum of one sweep launch from the committed ncu --set full
    capture of this configuration (profiles/ncu_traffic.json names the capture and its command; None if there is
    no capture -- DRAM counters cannot be read without a profiler, so this is the one number that is not live)."""
    try:
        with open(os.path.join(ROOT, "profiles", "ncu_traffic.json")) as f:
            return json.load(f).get(f"config{k}_{dtype}", {}).get("dram_bytes_per_sweep_launch")
    except OSError:
        return None


def measured_hbm_gbs():
    """Driver-measured HBM copy bandwidth (MEASURED_PEAKS.json), else the fallback of B200_PROFILING.md."""
    try:
        with open(os.path.join(ROOT, "MEASURED_PEAKS.json")) as f:
            return float(json.load(f)["hbm_gbs"]), "MEASURED_PEAKS.json"
    except (OSError, KeyError, ValueError):
        return 6650.0, "fallback (B200_PROFILING.md)"


def oracle_sample(W, k, budget_s, steps, cores=None):
    """Pick the largest replica of config k (same physical size, coarser grid) whose `steps` oracle
    iterations fit `budget_s` on this host; with cores > 1 the oracle runs threaded over bands (bit-identical)."""
    cores = max(1, min(os.cpu_count() or 1, 15)) if cores is None else cores
    full = W.config(k)
    grids = [(full.nx, full.ny, full.nz)]
    while max(grids[-1]) > 8:
        g = grids[-1]
        grids.append((max(g[0] // 2, 1), max(g[1] // 2, 1) if full.dim > 1 else 1, max(g[2] // 2, 1) if full.dim > 2 else 1))
    rate = 2.0e7 * cores                      # conservative guess [updates/s]; only sizes the sample
    for g in grids:
        p = W.config(k, grid=g)
        if p.updates_per_sweep * steps / rate <= budget_s:
            return p, g, cores
    return p, g, cores


def time_oracle(W, k, budget_s, steps=1, warmup=0, cores=None):
    import oracle
    p, grid, cores = oracle_sample(W, k, budget_s, steps + warmup, cores)
    r = oracle.RefSolver(p, threads=cores)
    r.iterate(warmup)
    t0 = time.perf_counter()
    r.iterate(steps)
    dt = time.perf_counter() - t0
    return {"value": p.updates_per_sweep * steps / dt, "unit": UNIT, "cores": cores, "kind": "oracle",
            "sample": f"{steps} source iteration(s) of config {k} on a {grid[0]}x{grid[1]}x{grid[2]} replica "
                      f"({p.updates_per_sweep:.3e} updates each), oracle on {cores} thread(s)"
                      + (" over bands" if cores > 1 else "")}, dt / steps, p


def run_reference(args, W):
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    cb, s_per_step, p = time_oracle(W, args.config, budget_s=150.0, steps=args.steps, warmup=args.warmup)
    line = {"impl": "reference", "metric": METRIC, "value": cb["value"], "unit": UNIT, "n_gpus": args.gpus,
            "steps": args.steps, "warmup": args.warmup, "ms_per_step": s_per_step * 1e3,
            "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
            "config": {"workload": f"configs[{args.config}] {p.name} (bounded sample, see cpu_baseline.sample)",
                       "grid": [p.nx, p.ny, p.nz], "bands": len(p.C), "directions": len(p.w)},
            "cpu_baseline": cb,
            "e2e": {"value": cb["value"], "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
            "gpu_launches": 0}
    print(json.dumps(line), flush=True)


class Ranks:
    """Replicas-only multi-GPU plumbing: one process per GPU, no data-path collective;
    the only exchanges are a barrier and the MAX of a timing scalar.  Works with nccl (GPU) and gloo (CPU tests)."""

    def __init__(self, backend="nccl", device=None):
        import torch.distributed as dist
        self.dist = dist
        self.world = int(os.environ.get("WORLD_SIZE", "1"))
        self.rank = int(os.environ.get("RANK", "0"))
        self.local = int(os.environ.get("LOCAL_RANK", "0"))
        self.device = device
        if self.world > 1 and not dist.is_initialized():
            kw = {"device_id": device} if (backend == "nccl" and device is not None) else {}
            dist.init_process_group(backend, **kw)

    def barrier(self):
        if self.world > 1:
            self.dist.barrier()

    def max(self, x):
        import torch
        t = torch.tensor([float(x)], dtype=torch.float64, device=self.device if self.device is not None else "cpu")
        if self.world > 1:
            self.dist.all_reduce(t, op=self.dist.ReduceOp.MAX)
        return float(t.item())

    def aggregate(self, units_per_rank, seconds_local):
        """whole-job throughput: all ranks' units / slowest rank's time"""
        return self.world * units_per_rank / self.max(seconds_local)

    def close(self):
        if self.world > 1 and self.dist.is_initialized():
            self.dist.destroy_process_group()


def run_ours(args, W):
    import torch
    import paper_2503_23657_b200 as bte

    local = int(os.environ.get("LOCAL_RANK", "0"))
    if not torch.cuda.is_available():
        raise SystemExit("bench.py needs a CUDA device: there is no CPU fallback (use --impl reference for the oracle)")
    torch.cuda.set_device(local)
    dev = torch.device("cuda", local)
    R = Ranks("nccl", dev)
    world, rank = R.world, R.rank

    def barrier():
        R.barrier()
        torch.cuda.synchronize()

    p = W.config(args.config)
    prec = {"config": p.precision, "f64": W.FP64, "f32": W.FP32_STORE_FP64_ACC}[args.precision]
    dtype = "f32" if prec == W.FP32_STORE_FP64_ACC else "f64"
    solver = bte.Solver(p, precision=prec, device=dev)
    K, Wm = args.steps, max(args.warmup, 3)
    upd = solver.updates_per_sweep
    # plain-ALU peak measured in this run (register-only FFMA2 / DFMA chains on every SM), before the timed region
    import microbench
    peak_measured, n_sms = microbench.measure_fma_peak(dtype, dev)

    # ---- device-resident timing: K iterations in one bte_iterate call (inputs already in HBM)
    solver.iterate(Wm)
    solver.set_sweep_timing(K)
    sampler = ClockSampler(local)
    barrier()
    sampler.start()
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    e0.record()
    solver.iterate(K)
    e1.record()
    barrier()
    clocks = sampler.stop()
    ms = R.max(e0.elapsed_time(e1))
    sweep_ms, sweep_n = solver.sweep_timing()
    solver.set_sweep_timing(0)
    eps = solver.residual()

    # ---- end to end through the C-ABI host-buffer call: every step uploads Q from pinned host memory,
    # runs one iteration and downloads dT into pinned host memory
    import numpy as np
    Qsrc = p.Q if p.Q is not None else np.zeros((p.nz, p.ny, p.nx))
    Qh = torch.from_numpy(np.ascontiguousarray(Qsrc, dtype=np.float64)).pin_memory()
    dTh = torch.empty(solver.shape, dtype=torch.float64).pin_memory()
    qh = torch.empty((3,) + solver.shape, dtype=torch.float64).pin_memory()
    for _ in range(3):
        solver.solve_host(Qh, 1, reset=False, out=(dTh, qh))
    barrier()
    t0 = time.perf_counter()
    for _ in range(K):
        solver.solve_host(Qh, 1, reset=False, out=(dTh, qh))
    barrier()
    e2e_s = R.max(time.perf_counter() - t0)

    conv = None
    if not args.no_converge and rank == 0:
        solver.solve_host(Qh, 0, reset=True, out=(dTh, None))
        torch.cuda.synchronize()
        t0, n = time.perf_counter(), 0
        while n < 20000:
            solver.iterate(25)
            n += 25
            if solver.residual()[0] <= 1e-8:
                break
        conv = {"eps_T_target": 1e-8, "iterations": n, "seconds": time.perf_counter() - t0,
                "eps_T": solver.residual()[0], "reached": solver.residual()[0] <= 1e-8,
                "what": "wall time of bte_iterate from dT = 0, bte_residual checked every 25 iterations (cap 20000)"}

    if rank == 0:
        sweep_avg_ms = sweep_ms / max(sweep_n, 1)
        achieved = upd * FLOP_PER_UPDATE / (sweep_avg_ms * 1e-3) / 1e12
        peak = PEAK_TFLOPS[dtype]
        info = solver.schedule_info()
        # both floors of the sweep launch AS BUILT: t_alu = algorithmic flop / derived FMA peak, t_hbm = DRAM bytes the
        # kernel actually moves (ncu capture of this configuration) / measured HBM copy bandwidth; the larger one binds
        traffic = ncu_traffic(args.config, dtype)
        hbm_gbs, hbm_src = measured_hbm_gbs()
        t_alu_ms = upd * FLOP_PER_UPDATE / (peak * 1e12) * 1e3
        t_hbm_ms = traffic / (hbm_gbs * 1e9) * 1e3 if traffic else None
        bound = "hbm" if (t_hbm_ms is not None and t_hbm_ms > t_alu_ms) else "alu"
        line = {"metric": METRIC, "value": world * upd * K / (ms * 1e-3), "unit": UNIT, "n_gpus": world,
                "steps": K, "warmup": Wm, "ms_per_step": ms / K, "higher_is_better": True, "scaling": "weak",
                "vs_baseline": None, "dtype": dtype, "data": "synthetic",
                "config": {"workload": f"configs[{args.config}] {p.name}", "grid": [p.nx, p.ny, p.nz],
                           "solid_cells": p.n_solid, "bands": len(p.C), "directions": len(p.w),
                           "updates_per_step": upd, "parallelism": "replicas" if world > 1 else "single",
                           "l2": f"working set {info['workspace_bytes'] / 1e6:.0f} MB > 126 MB L2 (no flush needed)"
                                 if info["workspace_bytes"] > 2 * 126e6 else "working set fits L2 (state is L2-resident by design)",
                           "eps_T_after_timed_steps": eps[0]},
                "clocks": clocks,
                "e2e": {"value": world * upd * K / e2e_s, "unit": UNIT, "h2d_bytes_per_step": Qh.numel() * 8,
                        "d2h_bytes_per_step": (dTh.numel() + qh.numel()) * 8,
                        "what": "bte_solve_host(Q pinned host -> 1 iteration -> dT and q pinned host) per step"},
                "gpu_launches": solver.launches_per_iteration * K,
                "roofline": {"bound": bound, "kernel": "bte2_sweep_kernel" if solver.kernel_path == 2 else "bte_sweep_kernel",
                             "achieved": achieved, "peak": peak,
                             "unit": "TFLOP/s", "frac": achieved / peak, "traffic": traffic,
                             "peak_source": "derived: 148 SMs x %d FMA/clk x 2 x 1.965 GHz (DESIGN.md)" % (128 if dtype == "f32" else 64),
                             "peak_measured": peak_measured, "frac_of_measured": achieved / peak_measured,
                             "peak_measured_source": "microbench/fma_peak.cu in this run: register-only %s chains, %d SMs, "
                                                     "SM clock %s MHz during the timed region" %
                                                     ("FFMA2" if dtype == "f32" else "DFMA", n_sms, clocks.get("sm_mhz")),
                             "t_alu_ms": t_alu_ms, "t_hbm_ms": t_hbm_ms,
                             "hbm": {"achieved_gbs": traffic / (sweep_avg_ms * 1e-3) / 1e9 if traffic else None,
                                     "peak_gbs": hbm_gbs, "peak_source": hbm_src,
                                     "frac": traffic / (sweep_avg_ms * 1e-3) / 1e9 / hbm_gbs if traffic else None,
                                     "algorithmic_bytes": ALGORITHMIC_BYTES.get(args.config)},
                             "ms_per_launch": sweep_avg_ms, "launches_timed": sweep_n,
                             "share_of_step": sweep_ms / ms if ms > 0 else None,
                             "wavefront_occupancy": upd / info["thread_slot_updates"]},
                }
        if conv:
            line["time_to_1e-8"] = conv
        if not args.no_cpu_baseline and world == 1:
            # the oracle as it stands: single thread first, then threaded over bands
            line["cpu_baseline"] = time_oracle(W, args.config, budget_s=12.0, steps=1, cores=1)[0]
            line["cpu_baseline_threads"] = time_oracle(W, args.config, budget_s=12.0, steps=1)[0]
        print(json.dumps(line), flush=True)
    R.close()


def main():
    args = parse()
    import workloads as W
    if args.impl == "reference":
        run_reference(args, W)
    else:
        run_ours(args, W)


if __name__ == "__main__":
    main()
