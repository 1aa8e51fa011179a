#!/usr/bin/env python
"""Benchmark of the far-field mobility product (BASELINE.json metric) on B200.

  python bench.py [--gpus N] [--steps K] [--warmup W] [--config c4] [--impl ours|reference]

One "step" is one pass of the whole hot path (a1-a8: sorts, real-space pair sum, spreading, forward
FFTs, k-space pass, inverse FFTs, gather, epilogue) over one seeded synthetic configuration.  At N=1 the
workload is c4 (N = 1e5, M = 256, P = 12), the configuration the metric is quoted on.  With N > 1 GPUs
the path does not shard (replicas only): every rank runs an independent replica
of the same product on its own GPU, no data-path collective; value = products of all ranks / max time.

Prints ONE JSON line (rank 0).  ``--impl reference`` times the CPU oracle (oracle/) instead.
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
sys.path.insert(0, ROOT)

METRIC = "SE far-field mobility products/sec"
UNIT = "products/s"


def measured_peaks():
    path = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(path):
        try:
            d = json.load(open(path))
            return float(d["hbm_gbs"]), "measured (MEASURED_PEAKS.json)"
        except Exception:
            pass
    return 6650.0, "fallback (B200_PROFILING.md)"


class ClockSampler:
    """nvidia-smi clocks and throttle reasons sampled DURING the timed region."""
    Q = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,clocks_event_reasons.hw_thermal_slowdown,"
         "clocks_event_reasons.sw_thermal_slowdown,clocks_event_reasons.sw_power_cap")

    def __init__(self, index=0):
        self.rows, self.proc, self.index = [], None, index

    def start(self):
        try:
            self.proc = subprocess.Popen(["nvidia-smi", f"--id={self.index}", f"--query-gpu={self.Q}", "--format=csv,noheader,nounits",
                                          "-lms", "100"], stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
            self.thread = threading.Thread(target=self._read, daemon=True)
            self.thread.start()
        except Exception:
            self.proc = None

    def _read(self):
        for line in self.proc.stdout:
            self.rows.append(line.strip())

    def stop(self):
        if self.proc is None:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        time.sleep(0.25)
        self.proc.terminate()
        try:
            self.proc.wait(timeout=2)
        except Exception:
            self.proc.kill()
        sm, mx, reasons = [], [], set()
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        for r in self.rows:
            f = [x.strip() for x in r.split(",")]
            if len(f) < 7:
                continue
            try:
                sm.append(float(f[0])); mx.append(float(f[1]))
            except ValueError:
                continue
            for n, v in zip(names, f[3:7]):
                if v.lower().startswith("active"):
                    reasons.add(n)
        return {"sm_mhz": statistics.median(sm) if sm else None, "sm_max_mhz": max(mx) if mx else None,
                "samples": len(sm), "reasons": sorted(reasons)}


def cpu_oracle_seconds(wl, repeats=1):
    """One full O2 product of the workload on the host cores, as the oracle stands."""
    import oracle as O
    O.build()
    best = float("inf")
    for _ in range(repeats):
        t0 = time.perf_counter()
        O.o2_apply(wl.pos, wl.radii, wl.L, wl.xi, wl.rc, wl.M, wl.P, wl.F, wl.T, wl.S)
        best = min(best, time.perf_counter() - t0)
    return best, O.num_threads()


def measure_config(name, dev, peak, steps):
    """Cold-path product of one more configuration (north_star: every config reported at 1 GPU): device-timed
    ms per product, stage times, algorithmic HBM fractions of the three grid kernels."""
    import torch
    import workloads as W
    import paper_1506_08481_b200 as pk
    wl = W.make_workload(name)
    plan = pk.SePlan(wl.N, wl.L, wl.radii, wl.xi, wl.rc, wl.M, wl.P, wl.eta0)
    t = lambda a: torch.tensor(np.ascontiguousarray(a), device=dev, dtype=torch.float64)
    pos, F, T, S = t(wl.pos), t(wl.F), t(wl.T), t(wl.S)
    U = torch.empty((wl.N, 3), device=dev, dtype=torch.float64)
    Om = torch.empty_like(U)
    E = torch.empty((wl.N, 5), device=dev, dtype=torch.float64)
    stream = torch.cuda.current_stream()
    for _ in range(3):
        plan.apply(pos, F, T, S, U, Om, E)
    torch.cuda.synchronize()
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    e0.record(stream)
    for _ in range(steps):
        plan.apply(pos, F, T, S, U, Om, E)
    e1.record(stream)
    torch.cuda.synchronize()
    ms = e0.elapsed_time(e1) / steps
    plan.set_flags(pk.SE_TIMING)
    stage = {k: 0.0 for k in pk.STAGE_NAMES}
    for _ in range(steps):
        plan.apply(pos, F, T, S, U, Om, E)
        for k, v in plan.timings().items():
            stage[k] += v / steps
    G = float(wl.M) ** 3
    Gc = float(wl.M) ** 2 * (wl.M // 2 + 1)
    alg = {"spread": 24.0 * G + 120.0 * wl.N, "kspace": 144.0 * Gc, "gather": 48.0 * G + 120.0 * wl.N}
    out = {"N": wl.N, "M": wl.M, "P": wl.P, "ms_per_step": ms, "products_per_s": 1e3 / ms, "ns_per_particle": 1e6 * ms / wl.N,
           "stages_ms": {k: round(v, 4) for k, v in stage.items()},
           "hbm_frac": {k: alg[k] / (stage[k] * 1e-3) / 1e9 / peak for k in alg}}
    plan.destroy()
    del pos, F, T, S, U, Om, E
    torch.cuda.empty_cache()
    return out


def run_reference(args, rank, world):
    """--impl reference: the CPU oracle timed on the host cores, rank 0 only."""
    if rank != 0:
        return
    import workloads as W
    wl = W.make_workload(args.config)
    for _ in range(args.warmup):
        cpu_oracle_seconds(wl)
    t0 = time.perf_counter()
    threads = 1
    for _ in range(args.steps):
        _, threads = cpu_oracle_seconds(wl)
    dt = time.perf_counter() - t0
    value = args.steps / dt
    line = {
        "impl": "reference", "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": args.gpus, "steps": args.steps,
        "warmup": args.warmup, "ms_per_step": 1e3 * dt / args.steps, "higher_is_better": True, "scaling": "weak",
        "vs_baseline": None, "dtype": "f64", "data": "synthetic",
        "ns_per_particle": 1e9 * dt / args.steps / wl.N,
        "config": {"workload": f"{args.config}: N={wl.N}, M={wl.M}, P={wl.P}, phi={wl.phi}, radii={wl.meta['radii']}",
                   "N": wl.N, "M": wl.M, "P": wl.P, "xi": wl.xi, "r_c": wl.rc},
        "cpu_baseline": {"value": value, "unit": UNIT, "cores": threads, "kind": "oracle",
                         "sample": f"full {args.config} product (oracle O2, gcc -O2 -fopenmp) per step"},
        "e2e": {"value": value, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0,
    }
    print(json.dumps(line), flush=True)


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=20)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--config", default="c4", choices=["c1", "c2", "c3", "c4", "c5"])
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-other-configs", action="store_true", help="skip the c1-c3, c5 lines of 'all_configs'")
    args = ap.parse_args()
    args.warmup = max(args.warmup, 3) if args.impl == "ours" else args.warmup

    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    local_rank = int(os.environ.get("LOCAL_RANK", "0"))

    if args.impl == "reference":
        run_reference(args, rank, world)
        return

    import torch
    import workloads as W
    import paper_1506_08481_b200 as pk

    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device (the product path has no CPU fallback)")
    torch.cuda.set_device(local_rank)
    dev = torch.device("cuda", local_rank)
    dist = None
    if world > 1:
        import torch.distributed as dist
        dist.init_process_group("nccl", device_id=dev)

    wl = W.make_workload(args.config)
    plan = pk.SePlan(wl.N, wl.L, wl.radii, wl.xi, wl.rc, wl.M, wl.P, wl.eta0)
    t = lambda a: torch.tensor(np.ascontiguousarray(a), device=dev, dtype=torch.float64)
    pos, F, T, S = t(wl.pos), t(wl.F), t(wl.T), t(wl.S)
    U = torch.empty((wl.N, 3), device=dev, dtype=torch.float64)
    Om = torch.empty_like(U)
    E = torch.empty((wl.N, 5), device=dev, dtype=torch.float64)
    stream = torch.cuda.current_stream()

    def barrier():
        if dist is not None:
            dist.barrier()
        torch.cuda.synchronize()

    # ---- device-resident timing: W warm-up steps, then exactly K steps between events on the launch stream ----
    plan.set_flags(0)
    for _ in range(args.warmup):
        plan.apply(pos, F, T, S, U, Om, E)
    barrier()
    sampler = ClockSampler(local_rank)
    if rank == 0:
        sampler.start()
        time.sleep(0.15)
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    barrier()
    e0.record(stream)
    for _ in range(args.steps):
        plan.apply(pos, F, T, S, U, Om, E)
    e1.record(stream)
    barrier()
    ms_total = e0.elapsed_time(e1)
    launches = plan.last_launch_count() * args.steps
    clocks = sampler.stop() if rank == 0 else None
    if dist is not None:
        tmax = torch.tensor([ms_total], device=dev, dtype=torch.float64)
        dist.all_reduce(tmax, op=dist.ReduceOp.MAX)
        ms_total = float(tmax.item())
    ms_step = ms_total / args.steps
    value = world * args.steps / (ms_total * 1e-3)

    # ---- warm path, reported beside the headline: positions fixed by se_plan_set_positions, a1 reduced to
    # refreshing the moments; the headline above is the cold path with the sorts ----
    plan.set_positions(pos)
    for _ in range(2):
        plan.apply(None, F, T, S, U, Om, E)
    barrier()
    w0, w1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    w0.record(stream)
    for _ in range(args.steps):
        plan.apply(None, F, T, S, U, Om, E)
    w1.record(stream)
    barrier()
    warm_ms = w0.elapsed_time(w1) / args.steps
    plan.set_positions(None)

    # ---- per-stage CUDA-event times (library events on the launch stream), averaged over K steps ----
    plan.set_flags(pk.SE_TIMING)
    stage = {k: 0.0 for k in pk.STAGE_NAMES}
    for _ in range(args.steps):
        plan.apply(pos, F, T, S, U, Om, E)
        for k, v in plan.timings().items():
            stage[k] += v / args.steps
    plan.set_flags(0)

    # ---- end to end through the C-ABI host entry point: pinned host buffers, H2D + D2H inside the timed region ----
    hp = lambda a: torch.tensor(np.ascontiguousarray(a), dtype=torch.float64).pin_memory().numpy()
    hpos, hF, hT, hS = hp(wl.pos), hp(wl.F), hp(wl.T), hp(wl.S)
    hU, hW, hE = hp(np.zeros((wl.N, 3))), hp(np.zeros((wl.N, 3))), hp(np.zeros((wl.N, 5)))
    for _ in range(2):
        plan.apply_host(hpos, hF, hT, hS, hU, hW, hE)
    barrier()
    t0 = time.perf_counter()
    for _ in range(args.steps):
        plan.apply_host(hpos, hF, hT, hS, hU, hW, hE)       # synchronises the stream before returning
    barrier()
    e2e_s = time.perf_counter() - t0
    if dist is not None:
        tm = torch.tensor([e2e_s], device=dev, dtype=torch.float64)
        dist.all_reduce(tm, op=dist.ReduceOp.MAX)
        e2e_s = float(tm.item())
    e2e_value = world * args.steps / e2e_s

    if rank != 0:
        if dist is not None:
            dist.destroy_process_group()
        return

    # ---- roofline of the dominant own kernel (cuFFT stages are library calls, reported separately) ----
    peak, peak_src = measured_peaks()
    G = float(wl.M) ** 3
    Gc = float(wl.M) ** 2 * (wl.M // 2 + 1)
    alg_bytes = {                                   # algorithmic bytes per launch
        "spread": 24.0 * G + 120.0 * wl.N,          # three grids written once + particle data
        "kspace": 144.0 * Gc,                       # 3 complex grids read, 6 written
        "gather": 48.0 * G + 120.0 * wl.N,          # six grids read once + particle data
    }
    own = {k: stage[k] for k in ("sort", "real", "spread", "kspace", "gather", "epilogue")}
    dom = max(("spread", "kspace", "gather"), key=lambda k: stage[k])
    achieved = alg_bytes[dom] / (stage[dom] * 1e-3) / 1e9
    # dram__bytes_read.sum + dram__bytes_write.sum per launch, from the ncu --set full capture summarised in
    # profiles/r01g_summary.md (c4 only; other configs have no capture)
    traffic_c4 = {"spread": 0.0895e9 + 352.0e6, "kspace": 0.4028e9 + 754.1e6, "gather": 1.4570e9 + 21.9e6}
    traffic = traffic_c4.get(dom) if args.config == "c4" else None
    # spreading and gather are FP64-issue bound before they are HBM bound: 12 N P^3 DFMA each
    try:
        fp64_peak = pk.measure_fp64_peak()
    except Exception:
        fp64_peak = None
    sg_flops = 2.0 * 12.0 * wl.N * float(wl.P) ** 3
    per_kernel = {}
    for k in alg_bytes:
        gbs = alg_bytes[k] / (stage[k] * 1e-3) / 1e9
        per_kernel[k] = {"ms": stage[k], "GB/s": gbs, "frac": gbs / peak}
        if k in ("spread", "gather"):
            tf = sg_flops / (stage[k] * 1e-3) / 1e12
            per_kernel[k]["fp64_TFLOP/s"] = tf
            per_kernel[k]["fp64_frac"] = tf / fp64_peak if fp64_peak else None
    roofline = {"kernel": dom, "bound": "hbm", "achieved": achieved, "peak": peak, "unit": "GB/s", "frac": achieved / peak,
                "traffic": traffic, "peak_source": peak_src, "fp64_peak_TFLOP/s": fp64_peak, "all": per_kernel}

    cpu = None
    if not args.no_cpu_baseline:
        sec, threads = cpu_oracle_seconds(wl)
        cpu = {"value": 1.0 / sec, "unit": UNIT, "cores": threads, "kind": "oracle",
               "sample": f"one full {args.config} product (oracle O2 as it stands, gcc -O2 -fopenmp), {sec:.2f} s"}

    others = {}
    if world == 1 and not args.no_other_configs and not args.no_cpu_baseline:
        for name in ("c1", "c2", "c3", "c5"):
            if name != args.config:
                try:
                    others[name] = measure_config(name, dev, peak, 5 if name == "c5" else args.steps)
                except Exception as exc:           # e.g. not enough memory on a shared device: reported, not fatal
                    others[name] = {"error": str(exc)[:200]}

    line = {
        "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps, "warmup": args.warmup,
        "ms_per_step": ms_step, "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f64",
        "data": "synthetic", "ns_per_particle": 1e6 * ms_step / wl.N,
        "config": {"workload": f"{args.config}: N={wl.N}, M={wl.M}, P={wl.P}, phi={wl.phi}, radii={wl.meta['radii']}, "
                               f"positions={wl.meta['positions']}", "N": wl.N, "M": wl.M, "P": wl.P, "xi": wl.xi, "r_c": wl.rc,
                   "parallelism": "replicas only" if world > 1 else "single GPU",
                   "l2": "no flush: per-step working set (grids + spectra) is %.1f GB >> 126 MB L2" % (plan.workspace_bytes() / 1e9)},
        "warm_ms_per_step": warm_ms, "stages_ms": stage, "fft_ms": stage["fft_fwd"] + stage["fft_inv"], "own_kernels_ms": sum(own.values()),
        "clocks": clocks,
        "e2e": {"value": e2e_value, "unit": UNIT, "h2d_bytes_per_step": 14 * 8 * wl.N, "d2h_bytes_per_step": 11 * 8 * wl.N,
                "ms_per_step": 1e3 * e2e_s / args.steps},
        "gpu_launches": launches,
        "roofline": roofline,
        "cpu_baseline": cpu,
        "all_configs": others,
    }
    print(json.dumps(line), flush=True)
    if dist is not None:
        dist.destroy_process_group()


if __name__ == "__main__":
    main()
