#!/usr/bin/env python
"""bench.py -- plans/s of the gL-BFGS hot path (BASELINE.json metric) on N B200s of one node.

A "step" is one pass of the whole hot path over one synthetic plan pool: gmco_create (a0),
gmco_optimize (a1-a7), gmco_result (a8), gmco_destroy.  The workload at N = 1 is BASELINE.json
configs[2] ("gMCO production": 252 dwell positions, 12000 points, K = 1000 plans, m = 10, 200
iterations) -- the configuration the metric ("at K = 1000") is quoted on.  With N > 1 every rank
optimises its own 1000-plan pool (plans are independent: K-sharding, no data-path collective,
weak scaling).

  python bench.py [--gpus N] [--steps K] [--warmup W] [--impl ours|reference] [--config C3]
                  [--precision tf32x3|simt]

Prints ONE JSON line on rank 0 (see DESIGN.md section 6 for every key).
"""
from __future__ import annotations

import argparse
import json
import os
import sys
import threading
import time
from pathlib import Path

import numpy as np

ROOT = Path(__file__).resolve().parent
sys.path.insert(0, str(ROOT))

import gmco_cases as gc  # noqa: E402

METRIC, UNIT = "plans_per_s", "plans/s"
# dram__bytes_read.sum + dram__bytes_write.sum per launch from `ncu --set full` captures: rows "config,kernel,read,write,source"
NCU_TRAFFIC_FILE = ROOT / "profiles" / "ncu_traffic.csv"


def ncu_traffic(config: str, kernel: str):
    """DRAM bytes per launch of `kernel` on `config` from the committed ncu summary, or None when there is no capture."""
    if not NCU_TRAFFIC_FILE.exists():
        return None
    for ln in NCU_TRAFFIC_FILE.read_text().splitlines():
        f = [v.strip() for v in ln.split(",")]
        if len(f) >= 4 and f[0] == config and f[1] == kernel:
            return int(float(f[2]) + float(f[3]))
    return None


def env_int(name, default):
    return int(os.environ.get(name, default))


def load_peaks():
    p = ROOT / "MEASURED_PEAKS.json"
    if p.exists():
        d = json.loads(p.read_text())
        return dict(hbm_gbs=d["hbm_gbs"], bf16_burst=d["bf16_tflops"], bf16_sustained=d["bf16_tflops_sustained"],
                    source="measured")
    return dict(hbm_gbs=6650.0, bf16_burst=1590.0, bf16_sustained=1400.0, source="fallback")


class ClockSampler:
    """SM clock and throttle reasons DURING the timed region (B200_PROFILING.md), read through NVML in a
    thread (two light queries per sample; a polling nvidia-smi process was seen to stall kernel launches)."""
    REASONS = (("hw_slowdown", 0x8), ("hw_thermal_slowdown", 0x40), ("sw_thermal_slowdown", 0x20),
               ("sw_power_cap", 0x4))

    def __init__(self, index, period_s=0.02):
        self.index, self.period, self.rows, self.stop, self.t, self.h = index, period_s, [], False, None, None

    def __enter__(self):
        if self.period <= 0:
            return self
        try:
            import pynvml
            pynvml.nvmlInit()
            vis = os.environ.get("CUDA_VISIBLE_DEVICES")
            phys = int(vis.split(",")[self.index]) if vis and vis.replace(",", "").isdigit() else self.index
            self.nv, self.h = pynvml, pynvml.nvmlDeviceGetHandleByIndex(phys)
            self.max = float(pynvml.nvmlDeviceGetMaxClockInfo(self.h, pynvml.NVML_CLOCK_SM))
            self._sample()                               # first call pays NVML's lazy set-up, outside the timed region
            self.rows.clear()
            self.t = threading.Thread(target=self._run, daemon=True)
            self.t.start()
        except Exception:                                # no NVML: the JSON line says so (samples = 0)
            self.h = None
        return self

    def _sample(self):
        sm = float(self.nv.nvmlDeviceGetClockInfo(self.h, self.nv.NVML_CLOCK_SM))
        try:
            mask = int(self.nv.nvmlDeviceGetCurrentClocksEventReasons(self.h))
        except Exception:
            mask = int(self.nv.nvmlDeviceGetCurrentClocksThrottleReasons(self.h))
        self.rows.append((sm, mask))

    def _run(self):
        while not self.stop:
            try:
                self._sample()
            except Exception:
                break
            time.sleep(self.period)

    def __exit__(self, *a):
        self.stop = True
        if self.t:
            self.t.join(timeout=2)

    def summary(self):
        if not self.rows:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": [], "samples": 0}
        reasons = sorted({n for _, m in self.rows for n, bit in self.REASONS if m & bit})
        return {"sm_mhz": float(np.median([r[0] for r in self.rows])), "sm_max_mhz": self.max, "reasons": reasons,
                "samples": len(self.rows)}


def oracle_leg(case, sample_plans):
    """The fp64 oracle as it stands on the host cores, on a bounded sample of the same workload."""
    import oracle
    oracle.build()
    w = case.weights[:sample_plans]
    t0 = time.perf_counter()
    oracle.optimize(case.D, case.structures, case.rx, case.T0, w, m=case.m, iters=case.iters)
    dt = time.perf_counter() - t0
    return sample_plans / dt, dt, oracle.num_threads()


def oracle_leg_one_core(case, n_plans=4):
    """The same oracle on ONE core: its only parallelism is OpenMP over plans, so a one-plan call runs on one thread."""
    import oracle
    oracle.build()
    t0 = time.perf_counter()
    for k in range(n_plans):
        oracle.optimize(case.D, case.structures, case.rx, case.T0, case.weights[k:k + 1], m=case.m, iters=case.iters)
    dt = time.perf_counter() - t0
    return n_plans / dt, dt


def measure_tf32_peak(torch, seconds=3.0):
    """Dense tf32 matmul throughput measured the way MEASURED_PEAKS.json measured bf16: torch.matmul 8192^3 (2 N^3 flops)
    with tf32 allowed, best of 10 (burst) and back to back for `seconds` (sustained), CUDA events."""
    n = 8192
    old = torch.backends.cuda.matmul.allow_tf32
    torch.backends.cuda.matmul.allow_tf32 = True
    try:
        a = torch.randn(n, n, device="cuda"); b = torch.randn(n, n, device="cuda"); c = torch.empty(n, n, device="cuda")
        for _ in range(3):
            torch.matmul(a, b, out=c)
        best = None
        for _ in range(10):
            e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            e0.record(); torch.matmul(a, b, out=c); e1.record(); e1.synchronize()
            best = e0.elapsed_time(e1) if best is None else min(best, e0.elapsed_time(e1))
        reps = max(10, int(seconds * 1e3 / best))
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        e0.record()
        for _ in range(reps):
            torch.matmul(a, b, out=c)
        e1.record(); e1.synchronize()
        flops = 2.0 * n ** 3
        return {"tf32_tflops": flops / (best * 1e-3) / 1e12, "tf32_tflops_sustained": flops * reps / (e0.elapsed_time(e1) * 1e-3) / 1e12,
                "how": f"torch.matmul fp32 inputs, allow_tf32, 8192^3: best of 10 (burst) and {reps} back to back (sustained), CUDA events"}
    finally:
        torch.backends.cuda.matmul.allow_tf32 = old


def run_reference(args, case):
    rank = env_int("RANK", 0)
    if rank != 0:
        return
    # bounded: about 12 s per step at 256 plans on 16 cores; with many steps the per-step sample shrinks so that the
    # whole --steps/--warmup run still ends within a few minutes (plans are independent: plans/s does not depend on it)
    total = max(args.warmup + args.steps, 1)
    sample = args.ref_sample if total <= 8 else max(16, args.ref_sample * 8 // total)
    sample = min(sample, case.n_plans)
    vals = []
    for i in range(args.warmup + args.steps):
        v, dt, cores = oracle_leg(case, sample)
        if i >= args.warmup:
            vals.append((v, dt))
    value = float(np.mean([v for v, _ in vals]))
    ms = float(np.mean([dt for _, dt in vals]) * 1e3)
    desc = f"{sample} of {case.n_plans} plans of {case.name}, full {case.iters} iterations, OpenMP over plans"
    print(json.dumps({
        "impl": "reference", "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": args.gpus, "steps": args.steps,
        "warmup": args.warmup, "ms_per_step": ms, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
        "dtype": "f64", "data": "synthetic", "plan_iterations_per_s": value * case.iters,
        "config": workload_config(case, args, None),
        "cpu_baseline": {"value": value, "unit": UNIT, "cores": cores, "kind": "oracle", "sample": desc},
        "e2e": {"value": value, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
    }))


def max_over_ranks_ms(ms: float, world: int, device) -> float:
    """The slowest rank's time: one all-reduce(MAX) of a scalar, outside every timed region."""
    if world == 1:
        return ms
    import torch
    import torch.distributed as dist
    t = torch.tensor([ms], dtype=torch.float64, device=device)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())


def job_value(plans_per_rank: int, world: int, steps: int, ms_max: float) -> float:
    """Whole-job plans/s: every rank optimises its own pool (weak scaling), time = max over ranks."""
    return world * plans_per_rank * steps / (ms_max * 1e-3)


def workload_config(case, args, stats):
    cfg = {"workload": f"{case.name}: BASELINE.json configs[{['C1','C2','C3','C4'].index(case.name)}]",
           "n_points": case.n_points, "n_dwell": case.n_dwell, "plans_per_gpu": case.n_plans, "m": case.m,
           "iters": case.iters, "step": "gmco_create + gmco_optimize + gmco_result + gmco_destroy",
           "l2": "flushed between timed steps (512 MiB write)", "parallelism": f"k-shard x{args.gpus}"}
    cfg["eps"] = getattr(args, "eps", 0.0)
    cfg["compaction"] = getattr(args, "compaction", 1)
    cfg["line_search"] = getattr(args, "line_search", 0)
    cfg["wide_accum"] = getattr(args, "wide_accum", 0)
    cfg["dose_kernel_option"] = getattr(args, "dose_kernel", 0)
    if stats:
        cfg["rounds"] = stats["rounds"]
        cfg["device_bytes"] = stats["device_bytes"]
        cfg["dose_kernel"] = stats.get("dose_kernel_name")
    return cfg


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=5)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--config", default="C3", choices=["C1", "C2", "C3", "C4"])
    ap.add_argument("--precision", default="tf32x3", choices=["tf32x3", "simt"])
    ap.add_argument("--ref-sample", type=int, default=256, help="plans per oracle step (bounded sample)")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-peak", action="store_true", help="skip the live tf32 matmul peak measurement (roofline falls back to the nominal ratio)")
    ap.add_argument("--dose-kernel", type=int, default=0, choices=[0, 1, 2], help="gmco_options.dose_kernel (1 = keep the single-CTA dose kernel; 2 = CTA pairs for the gradient contraction as well, an option that is off by default)")
    ap.add_argument("--line-search", type=int, default=0, choices=[0, 1], help="gmco_options.line_search (1 = polynomial line search, an option that is off by default)")
    ap.add_argument("--wide-accum", type=int, default=0, choices=[0, 1], help="gmco_options.wide_accum (1 = split main accumulator above 256 dwell positions)")
    ap.add_argument("--no-gsa", action="store_true", help="skip the gSA-vs-gL-BFGS comparison leg (C5)")
    ap.add_argument("--no-other-configs", action="store_true", help="skip the C1 / C2 / C4 legs (SURVEY 8(d): 'plus the same for C1, C2, C4')")
    ap.add_argument("--clock-period", type=float, default=0.02, help="seconds between NVML clock samples (0 = off)")
    ap.add_argument("--eps", type=float, default=0.0, help="per-plan stopping rule (PAPER.md:119); 0 = exactly `iters` iterations")
    ap.add_argument("--compaction", type=int, default=1, choices=[0, 1], help="gmco_options.compaction")
    ap.add_argument("--characterise", action="store_true",
                    help="add the K sweep (Fig. 4a/4b) and the eps sweep (Fig. 3a) legs, outside the timed region")
    args = ap.parse_args()
    args.warmup = max(args.warmup, 0)

    rank, world, local = env_int("RANK", 0), env_int("WORLD_SIZE", 1), env_int("LOCAL_RANK", 0)
    case = gc.make_case(args.config, seed_weights=7 + rank)

    if args.impl == "reference":
        run_reference(args, case)
        return

    import torch
    import torch.distributed as dist
    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device -- the product path has no CPU fallback")
    torch.cuda.set_device(local)
    if world > 1:
        dist.init_process_group("nccl", device_id=torch.device("cuda", local))

    from paper_1904_01567_b200 import build
    build.build()
    import paper_1904_01567_b200 as g

    prec = g.GMCO_PREC_TF32X3 if args.precision == "tf32x3" else g.GMCO_PREC_SIMT_FP32
    K, A, S, N = case.n_plans, case.n_dwell, case.n_structs, case.n_points
    stream = torch.cuda.current_stream()
    D_dev = torch.from_numpy(case.D).cuda(); T0_dev = torch.from_numpy(case.T0).cuda()
    w_dev = torch.from_numpy(case.weights).cuda()
    D_pin = torch.from_numpy(case.D).pin_memory(); T0_pin = torch.from_numpy(case.T0).pin_memory()
    w_pin = torch.from_numpy(case.weights).pin_memory()
    out_pin = {k: torch.empty(s, dtype=dt).pin_memory() for k, s, dt in
               (("T", (K, A), torch.float32), ("F", (K,), torch.float32), ("dvh", (K, S), torch.float32),
                ("terms", (K, S, 2), torch.float32), ("it", (K,), torch.int32), ("st", (K,), torch.int32))}
    out_dev = {k: torch.empty_like(v, device="cuda") for k, v in out_pin.items()}
    flush = torch.empty(512 << 20, dtype=torch.uint8, device="cuda")
    L = g.lib()
    last = {}

    def step(host: bool, profile: bool = False):
        Dm, Tm, wm, om = (D_pin, T0_pin, w_pin, out_pin) if host else (D_dev, T0_dev, w_dev, out_dev)
        opt = g.binding.make_options(m=case.m, precision=prec, eps=args.eps, compaction=args.compaction, dose_kernel=args.dose_kernel,
                                     line_search=args.line_search, wide_accum=args.wide_accum)
        h = g.gmco_create(Dm, case.structures, case.rx, opt, stream)
        try:
            if profile:
                g.gmco_set_profiling(h, True)
            g.gmco_optimize(h, Tm, wm, case.iters, stream)
            g.binding._check(L.gmco_result(h.ptr, om["T"].data_ptr(), om["F"].data_ptr(), om["dvh"].data_ptr(),
                                           om["terms"].data_ptr(), om["it"].data_ptr(), om["st"].data_ptr()), h)
            last["stats"] = g.gmco_get_stats(h)
            last["stats"]["dose_kernel_name"] = g.DOSE_KERNEL_NAMES.get(last["stats"]["dose_kernel"])
        finally:
            g.gmco_destroy(h)

    def timed(host, steps, profile=False):
        tot = 0.0
        for _ in range(steps):
            flush.fill_(1)                                   # evict L2 between timed steps
            e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            e0.record(stream); step(host, profile); e1.record(stream)
            e1.synchronize()
            tot += e0.elapsed_time(e1)
        return tot

    def barrier():
        torch.cuda.synchronize()
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    def max_over_ranks(ms):
        return max_over_ranks_ms(ms, world, "cuda")

    for _ in range(args.warmup):
        step(False); step(True)
    barrier()
    with ClockSampler(local, args.clock_period) as clk:
        ms_dev = timed(False, args.steps)
        barrier()
    ms_dev = max_over_ranks(ms_dev)
    stats = dict(last["stats"])
    barrier()
    ms_e2e = max_over_ranks(timed(True, args.steps))
    barrier()
    # roofline leg: same steps with per-launch CUDA events around the contraction kernel (in-library)
    prof = None
    if rank == 0:
        timed(False, min(args.steps, 3), profile=True)
        prof = dict(last["stats"])
    barrier()

    value = job_value(K, world, args.steps, ms_dev)
    e2e_value = job_value(K, world, args.steps, ms_e2e)
    h2d = case.D.nbytes + case.T0.nbytes + case.weights.nbytes
    d2h = sum(v.numel() * v.element_size() for v in out_pin.values())

    if rank == 0:
        peaks = load_peaks()
        line = {
            "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps, "warmup": args.warmup,
            "ms_per_step": ms_dev / args.steps, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
            "dtype": "tf32x3" if prec == g.GMCO_PREC_TF32X3 else "f32", "data": "synthetic",
            "plan_iterations_per_s": value * case.iters,
            "config": workload_config(case, args, stats),
            "e2e": {"value": e2e_value, "unit": UNIT, "h2d_bytes_per_step": int(h2d), "d2h_bytes_per_step": int(d2h),
                    "ms_per_step": ms_e2e / args.steps},
            "gpu_launches": int(stats["kernel_launches"] * args.steps),
            "clocks": clk.summary(),
            "paper_context": "gL-BFGS 0.9 ms/plan = ~1111 plans/s on a Titan X (Pascal), real cases, eps=1e-3 (PAPER.md:180)",
        }
        # Every leg below is auxiliary to the headline numbers above: a failure in one of them is recorded in the line
        # instead of costing the run its record.
        def leg(name, fn):
            try:
                return fn()
            except Exception as e:                              # noqa: BLE001 -- reported, not swallowed
                return {"error": f"{name}: {type(e).__name__}: {e}"}

        tf32 = None
        if not (args.no_peak or prec != g.GMCO_PREC_TF32X3):
            tf32 = leg("tf32 peak", lambda: measure_tf32_peak(torch))
            if "error" in tf32:
                line["tf32_peak_error"], tf32 = tf32["error"], None
        line["roofline"] = leg("roofline", lambda: roofline(case, prec, g, prof, peaks, tf32, clk.summary()))
        if not args.no_gsa:
            line["gsa_vs_glbfgs"] = leg("gsa", lambda: gsa_leg(g, torch, stream))
        if not args.no_other_configs:
            line["other_configs"] = leg("other configs", lambda: other_configs_leg(g, torch, stream, prec, case.name, not args.no_cpu_baseline))
        if args.characterise:
            line["characterisation"] = leg("characterise", lambda: characterise_leg(g, torch, stream, prec))
        if not args.no_cpu_baseline:
            def cpu():
                v, dt, cores = oracle_leg(case, args.ref_sample)
                v1, dt1 = oracle_leg_one_core(case)
                return {"value": v, "unit": UNIT, "cores": cores, "kind": "oracle",
                        "sample": f"{args.ref_sample} of {K} plans of {case.name}, full {case.iters} "
                                  f"iterations, {dt:.1f} s, OpenMP over plans",
                        "value_1core": v1, "sample_1core": f"4 plans one after the other, {dt1:.1f} s"}
            line["cpu_baseline"] = leg("cpu baseline", cpu)
        print(json.dumps(line))
    if world > 1:
        dist.destroy_process_group()


def characterise_leg(g, torch, stream, prec):
    """The paper's two characterisation experiments on the synthetic stand-in (C3 geometry, BASELINE.json configs[2]),
    outside the timed region of the headline metric; inputs resident in HBM, CUDA events, best of 2 after a warm-up.
    k_sweep  -- Fig. 4a/4b: optimisation time and device memory against the number of plans, gL-BFGS
                at eps = 1e-3 (the figure's "clinically useful" setting), 200-iteration cap.
    eps_sweep -- Fig. 3a: stopping criterion against optimisation time (speed-up normalised to
                eps = 1e-7) and the fraction of non-dominated plans over the individual objectives of Eq. 4 (one column per weighted
                term: configs[2] draws a hidden weight per term, so a weighted-sum optimum is Pareto-optimal in these
                columns), K = 1000."""
    def run(case, eps, iters, reps=3):
        D = torch.from_numpy(case.D).cuda(); T0 = torch.from_numpy(case.T0).cuda(); w = torch.from_numpy(case.weights).cuda()
        h = g.gmco_create(D, case.structures, case.rx, g.binding.make_options(m=case.m, precision=prec, eps=eps), stream)
        try:
            best = None
            for i in range(reps):
                e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
                e0.record(stream); g.gmco_optimize(h, T0, w, iters, stream); res = g.gmco_result(h); e1.record(stream)
                e1.synchronize()
                if i:
                    best = e0.elapsed_time(e1) if best is None else min(best, e0.elapsed_time(e1))
            stats = g.gmco_get_stats(h)
            # per-organ objectives of Eq. 4 WITHOUT the hidden weights: term / weight (unused sides are 0 / 0 -> 0)
            terms = res["objective_terms"].double().cpu().numpy()
            wts = case.weights.astype(np.float64)
            organ = np.where(wts > 0, terms / np.where(wts > 0, wts, 1.0), 0.0).reshape(len(wts), -1)
            organ = organ[:, (wts > 0).any(axis=0).reshape(-1)]        # the five weighted terms of configs[2]
            nd = g.gmco_pareto_front(h, organ.astype(np.float32), stream)["n_nondominated"]
        finally:
            g.gmco_destroy(h)
        it = res["iters_done"].cpu().numpy()
        return best, stats, it, nd

    k_sweep = []
    for K in (1, 10, 100, 1000, 10000):
        c = gc.make_case("C3", n_plans=K)
        ms, stats, it, _ = run(c, 1e-3, 200)
        k_sweep.append({"K": K, "ms": ms, "ms_per_plan": ms / K, "device_bytes": int(stats["device_bytes"]),
                        "rounds": int(stats["rounds"]), "mean_iters": float(it.mean())})
    eps_sweep = []
    c = gc.make_case("C3")
    for eps in (1e-7, 1e-6, 1e-5, 1e-4, 1e-3, 1e-2):
        ms, stats, it, nd = run(c, eps, 5000)
        eps_sweep.append({"eps": eps, "ms": ms, "rounds": int(stats["rounds"]), "mean_iters": float(it.mean()),
                          "max_iters": int(it.max()), "converged": int(stats["plans_converged"]),
                          "nondominated_fraction": nd / c.n_plans})
    for e in eps_sweep:
        e["speedup_vs_eps_1e-7"] = eps_sweep[0]["ms"] / e["ms"]
    return {"workload": "C3 geometry (12000 points x 252 dwell positions), weights log-uniform as in configs[2]",
            "k_sweep_eps_1e-3": k_sweep, "eps_sweep_K_1000": eps_sweep,
            "paper_context": "Fig. 4a: 0.9 ms/plan at 1000 plans, 10000 plans within 9 s, 2.6 GB at 10000 plans (PAPER.md:180, :228); "
                             "Fig. 3a: eps 1e-7 -> 1e-2 gives non-dominated 100 % -> 89.3 %, speed-up 1 -> 10, 99.3 % at 1e-3 "
                             "(PAPER.md:170); Titan X (Pascal), clinical cases"}


def other_configs_leg(g, torch, stream, prec, headline, with_oracle):
    """the metric "plus the same for C1, C2, C4".  Outside the timed region of the headline: one pool per
    configuration, inputs resident in HBM, CUDA events around create + optimize + result + destroy, best of 3 after a
    warm-up (C4: best of 2).  C1 and C2 also time the oracle IN FULL (every plan, every iteration) on the host cores;
    C4's oracle time is not taken here (hours of CPU work; the parity tests follow sampled plans)."""
    import oracle
    out = {}
    for name in ("C1", "C2", "C4"):
        if name == headline:
            continue
        c = gc.make_case(name)
        D = torch.from_numpy(c.D).cuda(); T0 = torch.from_numpy(c.T0).cuda(); w = torch.from_numpy(c.weights).cuda()
        best, stats = None, None
        for i in range(3 if name == "C4" else 4):
            e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            e0.record(stream)
            h = g.gmco_create(D, c.structures, c.rx, g.binding.make_options(m=c.m, precision=prec), stream)
            try:
                g.gmco_optimize(h, T0, w, c.iters, stream)
                g.gmco_result(h)
                stats = g.gmco_get_stats(h)
            finally:
                g.gmco_destroy(h)
            e1.record(stream); e1.synchronize()
            if i:
                best = e0.elapsed_time(e1) if best is None else min(best, e0.elapsed_time(e1))
        row = {"n_points": c.n_points, "n_dwell": c.n_dwell, "plans": c.n_plans, "iters": c.iters, "ms_per_pool": best,
               "plans_per_s": c.n_plans / (best * 1e-3), "plan_iterations_per_s": c.n_plans * c.iters / (best * 1e-3),
               "rounds": int(stats["rounds"]), "device_bytes": int(stats["device_bytes"]),
               "dose_kernel": g.DOSE_KERNEL_NAMES.get(stats["dose_kernel"])}
        if with_oracle and name in ("C1", "C2"):
            oracle.build()
            t0 = time.perf_counter()
            oracle.optimize(c.D, c.structures, c.rx, c.T0, c.weights, m=c.m, iters=c.iters)
            dt = time.perf_counter() - t0
            row["oracle_full_s"] = dt
            row["oracle_plans_per_s"] = c.n_plans / dt
            row["oracle_cores"] = oracle.num_threads()
        out[name] = row
    return out


def gsa_leg(g, torch, stream):
    """BASELINE.json configs[4] (C5): 100 gSA chains x 20000 steps on C1 geometry against gL-BFGS on the same
    weights -- final objectives and time-to-solution.  Outside the timed region of the
    headline metric; inputs resident in HBM; CUDA events; best of 3 after one warm-up."""
    c = gc.make_case("C1", n_plans=100)
    tau = float(c.T0[0])
    steps, iters = 20000, 200
    jdx, z, u = (torch.from_numpy(a).cuda() for a in gc.sa_draws(c.n_dwell, 100, steps, seed=15))
    T0, w = torch.from_numpy(c.T0).cuda(), torch.from_numpy(c.weights).cuda()
    h = g.gmco_create(c.D, c.structures, c.rx, g.binding.make_options(m=10), stream)

    def timed(fn):
        best, out = None, None
        for i in range(4):
            e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            e0.record(stream); out = fn(); e1.record(stream); e1.synchronize()
            if i:
                best = e0.elapsed_time(e1) if best is None else min(best, e0.elapsed_time(e1))
        return best, out

    def lbfgs():
        g.gmco_optimize(h, T0, w, iters, stream)
        return g.gmco_result(h)

    try:
        ms32, o32 = timed(lambda: g.gmco_sa_run(h, T0, w, jdx, z, u, tau, precision=g.GMCO_SA_FP32, stream=stream))
        ms64, o64 = timed(lambda: g.gmco_sa_run(h, T0, w, jdx, z, u, tau, precision=g.GMCO_SA_FP64, stream=stream))
        msl, ol = timed(lbfgs)
    finally:
        g.gmco_destroy(h)
    Fl = ol["objective"].double()
    return {"workload": "C5: BASELINE.json configs[4], 100 chains x 20000 steps vs 100 plans x 200 L-BFGS iterations, C1 geometry",
            "gsa_fp32_ms": ms32, "gsa_fp64_ms": ms64, "glbfgs_ms": msl,
            "gsa_chain_steps_per_s": 100 * steps / (ms32 * 1e-3),
            "time_ratio_gsa_over_glbfgs": ms32 / msl,
            "median_F_gsa_fp32_over_glbfgs": float((o32["objective"] / Fl).median()),
            "median_F_gsa_fp64_over_glbfgs": float((o64["objective"] / Fl).median()),
            "paper_context": "gL-BFGS up to 67x faster than gSA, objectives within 0.2-0.4 % (PAPER.md:160-162, :180; Titan X Pascal)"}


def roofline(case, prec, g, prof, peaks, tf32, clocks):
    """Per-kernel rooflines of one round, from CUDA events the library records around every kernel of the profiled steps
    (gmco_set_profiling).  The object itself describes the DOMINANT kernel (the dose kernel); `per_kernel` holds all three.
    Algorithmic work: dose kernel 2 N A flops per plan-evaluation (one D t), gradient
    kernel 2 N A (one D^T r) -- the 3xTF32 split issues 3x that on the tensor pipe, and `achieved` counts issued flops;
    step kernel (4 m A + 10 A) x 4 bytes per plan-round (S, Y read twice, one pair written, g / x / p traffic).
    Peak of the tensor kernels: dense tf32 matmul measured in this run the way MEASURED_PEAKS.json measured bf16 (burst:
    each kernel is timed alone by its own events and the step is far too short to reach the power cap); alternatives
    are listed beside it.  Peak of the step kernel: the measured HBM copy bandwidth."""
    if not prof or not prof.get("eval_launches"):
        return None
    n = prof["eval_launches"]
    plans = prof["eval_plans"] / n                       # running plans per round (all K until plans start to finish)
    ms_dose, ms_grad, ms_step = prof["dose_ms"] / n, prof["grad_ms"] / n, prof["step_ms"] / n
    flops = 2.0 * case.n_points * case.n_dwell * plans   # one contraction
    if prec != g.GMCO_PREC_TF32X3:
        peak = 148 * 128 * 2 * 1.965e9 / 1e12
        ach = 2 * flops / ((ms_dose + ms_grad) * 1e-3) / 1e12
        return {"bound": "alu", "kernel": "k_simt_dose + k_simt_grad", "achieved": ach, "peak": peak, "unit": "TFLOP/s",
                "frac": ach / peak, "avg_launch_ms": ms_dose + ms_grad, "launches": n,
                "peak_source": "148 SM x 128 fp32 lanes x 2 x 1.965 GHz", "traffic": None}
    sm_mhz = (clocks or {}).get("sm_mhz") or 1965.0
    alts = {"nominal_ratio_of_measured_bf16_burst": peaks["bf16_burst"] * (1.1 / 2.25),
            "nominal_ratio_of_measured_bf16_sustained": peaks["bf16_sustained"] * (1.1 / 2.25),
            "issue_limit_4096_flop_per_clk_per_sm_at_sampled_clock": 4096 * 148 * sm_mhz * 1e6 / 1e12,
            "nominal_dense_tf32": 1100.0}
    if tf32:
        peak, src = tf32["tf32_tflops"], "measured in this run: " + tf32["how"] + " (burst)"
        alts["measured_tf32_sustained"] = tf32["tf32_tflops_sustained"]
    else:
        peak, src = alts["nominal_ratio_of_measured_bf16_burst"], f"{peaks['source']} bf16 burst x 1.1/2.25 (nominal tf32:bf16; no live tf32 measurement)"
    dose_name = prof.get("dose_kernel_name") or "k_dose_tc"

    def tensor(kernel, ms):
        issued = 3.0 * flops / (ms * 1e-3) / 1e12
        return {"bound": "tensor", "kernel": kernel, "achieved": issued, "peak": peak, "unit": "TFLOP/s", "frac": issued / peak,
                "achieved_fp32_equivalent": issued / 3.0, "avg_launch_ms": ms,
                "traffic": ncu_traffic(case.name, kernel.split("<")[0])}
    step_bytes = (4 * case.m * case.n_dwell + 10 * case.n_dwell) * 4.0 * plans
    step = {"bound": "hbm", "kernel": "k_step", "achieved": step_bytes / (ms_step * 1e-3) / 1e9, "peak": peaks["hbm_gbs"],
            "unit": "GB/s", "frac": step_bytes / (ms_step * 1e-3) / 1e9 / peaks["hbm_gbs"], "avg_launch_ms": ms_step,
            "traffic": ncu_traffic(case.name, "k_step"),
            "note": "latency-bound: one warp per plan, 2 m dependent dot products (DESIGN.md 5.3)"}
    dose, grad = tensor(dose_name, ms_dose), tensor("k_grad_tc<16>", ms_grad)
    out = dict(dose)
    out.update({"launches": n, "plans_per_launch": plans, "peak_source": src, "peak_alternatives": alts,
                "traffic_source": str(NCU_TRAFFIC_FILE.relative_to(ROOT)) if NCU_TRAFFIC_FILE.exists() else None,
                "round_ms": {"dose": ms_dose, "grad": ms_grad, "step": ms_step},
                "per_kernel": {"dose": dose, "grad": grad, "step": step}})
    return out


if __name__ == "__main__":
    main()
