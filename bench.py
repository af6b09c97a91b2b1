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
# dram__bytes_read.sum + dram__bytes_write.sum of one dose launch (k_dose_tc_pair, profiles/r1_ncu_dose_pair.md) + one
# k_grad_tc launch (profiles/r1_ncu_full_summary.md), from ncu --set full captures (constants copied from those files)
NCU_TRAFFIC_BYTES = {"C3": int((26.057472 + 3.099904 + 74.339328 + 4.086272) * 1e6)}   # cold-cache capture: ncu flushes L2 per kernel


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
    if stats:
        cfg["rounds"] = stats["rounds"]
        cfg["device_bytes"] = stats["device_bytes"]
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
    ap.add_argument("--no-gsa", action="store_true", help="skip the gSA-vs-gL-BFGS comparison leg (C5)")
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
        opt = g.binding.make_options(m=case.m, precision=prec, eps=args.eps, compaction=args.compaction)
        h = g.gmco_create(Dm, case.structures, case.rx, opt, stream)
        try:
            if profile:
                g.gmco_set_profiling(h, True)
            g.gmco_optimize(h, Tm, wm, case.iters, stream)
            g.binding._check(L.gmco_result(h.ptr, om["T"].data_ptr(), om["F"].data_ptr(), om["dvh"].data_ptr(),
                                           om["terms"].data_ptr(), om["it"].data_ptr(), om["st"].data_ptr()), h)
            last["stats"] = g.gmco_get_stats(h)
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
        line["roofline"] = roofline(case, prec, g, prof, peaks)
        if not args.no_gsa:
            line["gsa_vs_glbfgs"] = gsa_leg(g, torch, stream)
        if args.characterise:
            line["characterisation"] = characterise_leg(g, torch, stream, prec)
        if not args.no_cpu_baseline:
            v, dt, cores = oracle_leg(case, args.ref_sample)
            line["cpu_baseline"] = {"value": v, "unit": UNIT, "cores": cores, "kind": "oracle",
                                    "sample": f"{args.ref_sample} of {K} plans of {case.name}, full {case.iters} "
                                              f"iterations, {dt:.1f} s, OpenMP over plans"}
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


def roofline(case, prec, g, prof, peaks):
    """Dominant kernel = the contraction (fused dose+penalty+gradient) kernel.
    Algorithmic flops per launch = 4 N A K (one D t and one D^T r per plan); the 3xTF32
    split issues 3x that on the tensor pipe.  Peak: measured bf16 (sustained: the kernel runs inside a
    long step) x the guide's nominal tf32/bf16 ratio 1.1/2.25; SIMT: 148 SM x 128 lanes x 2 x 1.965 GHz."""
    if not prof or not prof.get("eval_launches"):
        return None
    # plan-evaluations per launch: the running plans of each round (all K until plans start to finish)
    plans_per_launch = prof["eval_plans"] / prof["eval_launches"]
    flops = 4.0 * case.n_points * case.n_dwell * plans_per_launch
    ms = prof["eval_ms"] / prof["eval_launches"]
    if prec == g.GMCO_PREC_TF32X3:
        peak = peaks["bf16_sustained"] * (1.1 / 2.25)
        issued = 3.0 * flops / (ms * 1e-3) / 1e12
        return {"bound": "tensor", "kernel": "dose + gradient contractions of one round (k_dose_tc_pair, or k_dose_tc where the pair kernel does not apply, + k_grad_tc), timed as a pair",
                "achieved": issued, "peak": peak, "unit": "TFLOP/s", "frac": issued / peak,
                "achieved_fp32_equivalent": issued / 3.0, "avg_launch_ms": ms, "launches": prof["eval_launches"],
                "plans_per_launch": plans_per_launch,
                "peak_source": f"{peaks['source']} bf16 sustained x 1.1/2.25 (nominal tf32:bf16)",
                "traffic": NCU_TRAFFIC_BYTES.get(case.name)}
    peak = 148 * 128 * 2 * 1.965e9 / 1e12
    ach = flops / (ms * 1e-3) / 1e12
    return {"bound": "alu", "kernel": "k_simt_dose + k_simt_grad", "achieved": ach, "peak": peak, "unit": "TFLOP/s",
            "frac": ach / peak, "avg_launch_ms": ms, "launches": prof["eval_launches"],
            "peak_source": "148 SM x 128 fp32 lanes x 2 x 1.965 GHz", "traffic": None}


if __name__ == "__main__":
    main()
