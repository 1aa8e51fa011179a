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


def config_dict(name, wl, world):
    """The `config` object of the JSON line; identical in both arms (--impl ours / reference)."""
    return {"workload": f"{name}: N={wl.N}, M={wl.M}, P={wl.P}, phi={wl.phi}, radii={wl.meta['radii']}, "
                        f"positions={wl.meta['positions']}", "N": wl.N, "M": wl.M, "P": wl.P, "xi": wl.xi, "r_c": wl.rc,
            "parallelism": "replicas only" if world > 1 else "single GPU",
            "l2": "no flush: the per-step working set (grids + spectra, > 2 GB at c4) is far larger than the 126 MB L2"}


def load_counters():
    """ncu counters of the own kernels (profiles/r02_counters.json, written from the tracked capture by
    `python -m paper_1506_08481_b200.profile_counters`); None when the file is absent."""
    path = os.path.join(ROOT, "profiles", "r02_counters.json")
    try:
        return json.load(open(path))
    except Exception:
        return None


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
    stream = torch.cuda.Stream()             # not the legacy default stream: the plan-owned CUDA graph (M <= 128) needs a capturable one
    torch.cuda.synchronize()
    for _ in range(3):
        plan.apply(pos, F, T, S, U, Om, E, stream=stream)
    torch.cuda.synchronize()
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    e0.record(stream)
    for _ in range(steps):
        plan.apply(pos, F, T, S, U, Om, E, stream=stream)
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


def real_pairs(wl):
    """Ordered pairs with minimum-image distance below r_c (the work of the real-space kernel), counted with a k-d tree."""
    try:
        from scipy.spatial import cKDTree
        pos = np.mod(wl.pos, wl.L)
        pos[pos >= wl.L] = 0.0
        t = cKDTree(pos, boxsize=wl.L)
        return float(t.count_neighbors(t, wl.rc) - wl.N)          # ordered pairs, self pairs removed
    except Exception:
        return float("nan")


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
        "config": config_dict(args.config, wl, world),
        "cpu_baseline": {"value": value, "unit": UNIT, "cores": threads, "kind": "oracle",
                         "sample": f"full {args.config} product per step (oracle O2 as it stands, gcc -O2 -fopenmp; its spreading "
                                   "loop and line FFTs are serial, only the gather, k-space and real-space loops are threaded)"},
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
    ap.add_argument("--real-overlap", type=int, default=None, choices=[0, 1, 2],
                    help="SE_OPT_REAL_OVERLAP of the plan (default: the library's); 0 runs the real-space kernel alone, one CTA per cell")
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
    if args.real_overlap is not None:
        plan.set_option(pk.SE_OPT_REAL_OVERLAP, args.real_overlap)
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
    ev = [torch.cuda.Event(enable_timing=True) for _ in range(args.steps + 1)]
    barrier()
    ev[0].record(stream)
    for k in range(args.steps):
        plan.apply(pos, F, T, S, U, Om, E)
        ev[k + 1].record(stream)
    barrier()
    ms_total = ev[0].elapsed_time(ev[-1])
    ms_median = statistics.median(ev[k].elapsed_time(ev[k + 1]) for k in range(args.steps))
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

    # ---- several right-hand sides on the cached configuration: products/s per batch size ----
    batch = {}
    plan.set_positions(pos)
    for nrhs in (1, 4, 8):
        Fb, Tb, Sb = F.repeat(nrhs, 1, 1), T.repeat(nrhs, 1, 1), S.repeat(nrhs, 1, 1)
        Ub, Wb, Eb = torch.empty_like(Fb), torch.empty_like(Fb), torch.empty_like(Sb)
        plan.apply_batch(None, Fb, Tb, Sb, Ub, Wb, Eb)
        barrier()
        b0, b1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        reps = max(1, args.steps // nrhs)
        b0.record(stream)
        for _ in range(reps):
            plan.apply_batch(None, Fb, Tb, Sb, Ub, Wb, Eb)
        b1.record(stream)
        barrier()
        ms_b = b0.elapsed_time(b1) / reps
        batch[f"nrhs{nrhs}"] = {"ms_per_batch": ms_b, "ms_per_rhs": ms_b / nrhs, "products_per_s": 1e3 * nrhs / ms_b}
        del Fb, Tb, Sb, Ub, Wb, Eb
    plan.set_positions(None)

    # ---- per-stage CUDA-event times (library events on the launch stream), averaged over K steps ----
    plan.set_flags(pk.SE_TIMING)
    samples = {k: [] for k in pk.STAGE_NAMES}
    for _ in range(args.steps):
        plan.apply(pos, F, T, S, U, Om, E)
        for k, v in plan.timings().items():
            samples[k].append(v)
    stage = {k: statistics.median(v) for k, v in samples.items()}          # median over the timed steps
    plan.set_flags(0)

    # ---- the other size-effect variants and the single-precision mesh, same workload, cold products.  They change
    # the discretisation (or the precision), so they are reported beside the headline, never as it. ----
    variants = {}
    if world == 1 and not args.no_other_configs:
        for key, opts, reps in (("real_space", {pk.SE_OPT_SIZE_VARIANT: 1}, args.steps), ("wave_space", {pk.SE_OPT_SIZE_VARIANT: 2}, max(2, args.steps // 5)),
                                ("fp32_mesh", {pk.SE_OPT_GRID_FP32: 1}, args.steps), ("real_space_fp32_mesh", {pk.SE_OPT_SIZE_VARIANT: 1, pk.SE_OPT_GRID_FP32: 1}, args.steps)):
            try:
                for k, v in opts.items():
                    plan.set_option(k, v)
                for _ in range(2):
                    plan.apply(pos, F, T, S, U, Om, E)
                barrier()
                v0, v1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
                v0.record(stream)
                for _ in range(reps):
                    plan.apply(pos, F, T, S, U, Om, E)
                v1.record(stream)
                barrier()
                variants[key] = {"ms_per_step": v0.elapsed_time(v1) / reps, "gpu_launches": plan.last_launch_count()}
            except Exception as exc:               # e.g. the 24 extra spectra of the wave-space variant do not fit
                variants[key] = {"error": str(exc)[:200]}
            finally:
                plan.set_option(pk.SE_OPT_SIZE_VARIANT, 0)
                plan.set_option(pk.SE_OPT_GRID_FP32, 0)

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
    e2e_sync_value = world * args.steps / e2e_s
    e2e_sync_ms = 1e3 * e2e_s / args.steps

    # ---- the same as a pipeline: the caller's copies on two copy streams, far_mobility_apply on a compute stream, device input and
    # output buffers double-buffered, so that the copies of the neighbouring steps overlap this step's kernels.  Every step still
    # copies its inputs from pinned host memory and its results back inside the timed region; events order upload -> product ->
    # download per buffer set, and a set is reused only after the step that used it has left it. ----
    e2e_mode = ("pipeline: uploads, far_mobility_apply and downloads on three streams, device buffers double-buffered "
                "(cudaMemcpyAsync from / to pinned host memory every step)")
    tp = lambda a: torch.tensor(np.ascontiguousarray(a), dtype=torch.float64).pin_memory()
    th_in = [tp(wl.pos), tp(wl.F), tp(wl.T), tp(wl.S)]
    th_out = [[tp(np.zeros((wl.N, k))) for k in (3, 3, 5)] for _ in range(2)]
    td_in = [[torch.empty_like(h, device=dev) for h in th_in] for _ in range(2)]
    td_out = [[torch.empty((wl.N, k), device=dev, dtype=torch.float64) for k in (3, 3, 5)] for _ in range(2)]
    s_up, s_run, s_down = torch.cuda.Stream(), torch.cuda.Stream(), torch.cuda.Stream()
    ev_up = [torch.cuda.Event() for _ in range(2)]
    ev_run = [torch.cuda.Event() for _ in range(2)]
    ev_down = [torch.cuda.Event() for _ in range(2)]

    def pipelined(n):
        for i in range(n):
            j = i & 1
            if i >= 2:
                s_up.wait_event(ev_run[j])                     # the product two steps ago has read these input buffers
            with torch.cuda.stream(s_up):
                for d, h in zip(td_in[j], th_in):
                    d.copy_(h, non_blocking=True)
            ev_up[j].record(s_up)
            s_run.wait_event(ev_up[j])
            if i >= 2:
                s_run.wait_event(ev_down[j])                   # its results have left these output buffers
            plan.apply(*td_in[j], *td_out[j], stream=s_run)
            ev_run[j].record(s_run)
            s_down.wait_event(ev_run[j])
            with torch.cuda.stream(s_down):
                for h, d in zip(th_out[j], td_out[j]):
                    h.copy_(d, non_blocking=True)
            ev_down[j].record(s_down)
            if i >= 1:
                ev_down[j ^ 1].synchronize()                   # host pacing: the previous step's results are on the host
        torch.cuda.synchronize()

    pipelined(4)
    barrier()
    t0 = time.perf_counter()
    pipelined(args.steps)
    barrier()
    e2e_s = time.perf_counter() - t0
    if dist is not None:
        tm = torch.tensor([e2e_s], device=dev, dtype=torch.float64)
        dist.all_reduce(tm, op=dist.ReduceOp.MAX)
        e2e_s = float(tm.item())
    e2e_value = world * args.steps / e2e_s
    # the pipeline's results against the synchronous entry point's (same product; equal to summation order)
    e2e_outputs_diff = max(float(np.abs(a.numpy() - b).max() / np.abs(b).max()) for a, b in zip(th_out[(args.steps - 1) & 1], (hU, hW, hE)))
    del td_in, td_out

    if rank != 0:
        if dist is not None:
            dist.destroy_process_group()
        return

    # ---- roofline of the dominant own kernel (stage times above: CUDA events of the library on the launch stream) ----
    # Algorithmic work per launch: bytes of the three grid kernels, useful FP64 operations of the
    # three arithmetic-bound ones.  `traffic` and the DFMA counts come from the tracked ncu capture
    # (profiles/r02_counters.json), never from literals here; absent file or other config -> null.
    peak, peak_src = measured_peaks()
    NOMINAL_HBM = 8000.0
    G = float(wl.M) ** 3
    Gc = float(wl.M) ** 2 * (wl.M // 2 + 1)
    alg_bytes = {
        "spread": 24.0 * G + 120.0 * wl.N,          # three grids written once + particle data
        "kspace": 144.0 * Gc,                       # 3 complex grids read, 6 written (x transforms fused in, no extra traffic)
        "gather": 48.0 * G + 120.0 * wl.N,          # six grids read once + particle data
    }
    try:
        fp64_peak = pk.measure_fp64_peak()
    except Exception:
        fp64_peak = None
    npairs = real_pairs(wl)
    alg_flops = {
        "spread": 2.0 * 12.0 * wl.N * float(wl.P) ** 3,      # 12 DFMA per particle and support point
        "gather": 2.0 * 12.0 * wl.N * float(wl.P) ** 3,
        "real": 600.0 * npairs,                              # ~600 FP64 instructions per ordered pair
    }
    counters = load_counters() if args.config == "c4" else None
    kname = {"spread": "k_spread", "gather": "k_gather", "kspace": "k_xmid", "real": "k_real"}

    def ncu(kind, key):
        try:
            return counters["kernels"][kname[kind]][key]
        except Exception:
            return None

    per_kernel = {}
    for k in ("spread", "gather", "kspace", "real"):
        e = {"ms": stage[k]}
        if k in alg_bytes:
            gbs = alg_bytes[k] / (stage[k] * 1e-3) / 1e9
            e.update({"GB/s": gbs, "hbm_frac_measured_peak": gbs / peak, "hbm_frac_nominal_8TBs": gbs / NOMINAL_HBM})
            rd, wr = ncu(k, "dram_bytes_read"), ncu(k, "dram_bytes_write")
            e["traffic"] = (rd + wr) if rd is not None and wr is not None else None
        if k in alg_flops:
            tf = alg_flops[k] / (stage[k] * 1e-3) / 1e12
            e.update({"fp64_TFLOP/s": tf, "fp64_frac": tf / fp64_peak if fp64_peak else None,
                      "fp64_pipe_busy_pct_ncu": ncu(k, "fp64_pipe_active_pct")})
        per_kernel[k] = e
    own = {k: stage[k] for k in ("sort", "real", "spread", "kspace", "gather", "epilogue")}
    dom = max(("spread", "kspace", "gather", "real"), key=lambda k: stage[k])
    if dom in ("spread", "gather", "real"):         # FP64-issue bound before HBM bound: report against the FP64 peak
        achieved = alg_flops[dom] / (stage[dom] * 1e-3) / 1e12
        roofline = {"kernel": dom, "bound": "alu", "achieved": achieved, "peak": fp64_peak, "unit": "TFLOP/s",
                    "frac": achieved / fp64_peak if fp64_peak else None, "traffic": per_kernel[dom].get("traffic"),
                    "peak_source": "measured on this run: independent DFMA chains (se_measure_fp64_peak); nominal 148 SM x 64 DFMA/clk x 2 x 1.965 GHz = 37.2"}
    else:
        achieved = alg_bytes[dom] / (stage[dom] * 1e-3) / 1e9
        roofline = {"kernel": dom, "bound": "hbm", "achieved": achieved, "peak": peak, "unit": "GB/s", "frac": achieved / peak,
                    "traffic": per_kernel[dom].get("traffic"), "peak_source": peak_src}
    roofline.update({"hbm_peak_GB/s": peak, "hbm_peak_source": peak_src, "hbm_nominal_GB/s": NOMINAL_HBM, "fp64_peak_TFLOP/s": fp64_peak,
                     "counters": "profiles/r02_counters.json" if counters else None, "all": per_kernel})

    cpu = None
    if not args.no_cpu_baseline:
        import oracle as O
        sec, threads = cpu_oracle_seconds(wl)
        parts = {}
        for nm, fl in (("real", O.PART_REAL), ("wave", O.PART_WAVE)):
            t0 = time.perf_counter()
            O.o2_apply(wl.pos, wl.radii, wl.L, wl.xi, wl.rc, wl.M, wl.P, wl.F, wl.T, wl.S, parts=fl)
            parts[nm] = time.perf_counter() - t0
        cpu = {"value": 1.0 / sec, "unit": UNIT, "cores": threads, "kind": "oracle", "stage_seconds": parts,
               "sample": f"one full {args.config} product (oracle O2 as it stands, gcc -O2 -fopenmp), {sec:.2f} s; real-space part alone "
                         f"{parts['real']:.2f} s, wave-space part alone {parts['wave']:.2f} s; the oracle's spreading loop and line FFTs are "
                         "serial, only its gather, k-space and real-space loops use the cores"}

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
        "ms_per_step_median": ms_median,
        "config": config_dict(args.config, wl, world),
        "workspace_GB": plan.workspace_bytes() / 1e9,
        "warm_ms_per_step": warm_ms, "batch_cached_positions": batch, "stages_ms": stage, "fft_ms": stage["fft_fwd"] + stage["fft_inv"], "own_kernels_ms": sum(own.values()),
        "clocks": clocks,
        "e2e": {"value": e2e_value, "unit": UNIT, "h2d_bytes_per_step": 14 * 8 * wl.N, "d2h_bytes_per_step": 11 * 8 * wl.N,
                "ms_per_step": 1e3 * e2e_s / args.steps,
                "mode": e2e_mode,
                "max_rel_diff_to_the_synchronous_call": e2e_outputs_diff,
                "one_at_a_time": {"value": e2e_sync_value, "ms_per_step": e2e_sync_ms,
                                  "mode": "far_mobility_apply_host, synchronises after every product"}},
        "gpu_launches": launches,
        "roofline": roofline,
        "cpu_baseline": cpu,
        "size_variants": variants,
        "all_configs": others,
    }
    print(json.dumps(line), flush=True)
    if dist is not None:
        dist.destroy_process_group()


if __name__ == "__main__":
    main()
