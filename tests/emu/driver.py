"""Runs libgmco's kernel SOURCE on the CPU emulation (tests/emu/_build/libgmco_emu.so) and reports, as one JSON line,
how the results compare with the fp64 oracle.  TEST INFRASTRUCTURE ONLY; started as a subprocess by
tests/test_emu_*.py so that the real library loaded by the other tests is untouched:

    python tests/emu/driver.py '<json: {"scenario": name, ...options}>'

Everything goes through the product's own Python binding (paper_1904_01567_b200.binding) pointed at the emulated
library: same C ABI, same host code, same kernels; only the PTX layer and the CUDA runtime are the models of
tests/emu/emu_ptx.h and emu_runtime.cc.
"""
from __future__ import annotations

import ctypes as C
import json
import sys
import time
from pathlib import Path

import numpy as np

ROOT = Path(__file__).resolve().parents[2]
sys.path.insert(0, str(ROOT))

import gmco_cases as gc  # noqa: E402
import oracle  # noqa: E402
import paper_1904_01567_b200.binding as b  # noqa: E402


def load(lib: Path):
    b.lib_path = lambda: lib
    b._lib = None
    b._stream = lambda stream: None          # no torch, no CUDA stream: the emulated runtime has one order of execution
    import paper_1904_01567_b200 as g
    E = C.CDLL(str(lib))
    E.emu_violation_message.restype = C.c_char_p
    E.emu_set.argtypes = [C.c_char_p, C.c_long]
    E.emu_counter.argtypes = [C.c_char_p]
    E.emu_counter.restype = C.c_long
    E.emu_traffic.argtypes = [C.c_char_p, C.c_int]
    E.emu_traffic.restype = C.c_long
    return g, E


def configure(E, a):
    for key in ("seed", "max_delay", "mma_delay", "dyn_misalign", "sm_count", "shuffle", "verbose", "starve_mask", "starve_period"):
        if key in a:
            E.emu_set(key.encode(), int(a[key]))


def custom_case(a):
    """C1 by default; any field of gmco_cases.make_case may be overridden from the scenario's arguments."""
    kw = {k: a[k] for k in ("n_plans", "n_cath", "n_pos", "counts", "m", "iters", "seed_points", "seed_weights") if k in a}
    return gc.make_case(a.get("case", "C1"), **kw)


def spread_start(c, seed=100):
    """Non-converged evaluation points (as tests/test_gpu_zy_fullsize.py): a random start scaled per plan over 0.5 .. 1.5."""
    return np.repeat(gc.random_starts(c, 1, seed=seed), c.n_plans, axis=0) * np.linspace(0.5, 1.5, c.n_plans)[:, None].astype(np.float32)


def eval_errors(out, ref):
    # a plan without any penalty has F = 0 and g = 0 exactly on both sides: compare those absolutely
    tiny = np.finfo(np.float64).tiny
    e_d = float((np.abs(out["dose"] - ref["dose"]) / np.abs(ref["dose"])).max())
    e_f = float((np.abs(out["F"] - ref["F"]) / np.maximum(ref["F"], tiny)).max())
    e_g = float((np.linalg.norm(out["grad_x"] - ref["grad_x"], axis=1) / np.maximum(np.linalg.norm(ref["grad_x"], axis=1), tiny)).max())
    return dict(dose=e_d, F=e_f, grad=e_g)


def options(a, c):
    kw = {k: a[k] for k in ("precision", "eps", "compaction", "dose_kernel", "wide_accum", "line_search", "eps_f", "max_trials") if k in a}
    return b.make_options(m=c.m, **kw)


def digest(*arrays):
    import hashlib
    h = hashlib.sha256()
    for x in arrays:
        h.update(np.ascontiguousarray(x).tobytes())
    return h.hexdigest()


def report(E, **kw):
    kw.update(violations=int(E.emu_violations()), violation=(E.emu_violation_message() or b"").decode(),
              hangs=int(E.emu_counter(b"hangs")), mma=int(E.emu_counter(b"mma")), tma=int(E.emu_counter(b"tma")),
              live_allocations=int(E.emu_live_allocations()))
    return kw


# ---- scenarios -----------------------------------------------------------------------------------------------------
def sc_evaluate(g, E, a):
    """One gmco_evaluate: dose, objective and gradient of every plan against the oracle."""
    c = custom_case(a)
    T = spread_start(c) if a.get("start", "spread") == "spread" else np.repeat(c.T0[None], c.n_plans, axis=0)
    ref = oracle.evaluate(c.D, c.structures, T, c.weights)
    sched = g.gmco_tc_schedule(c.n_dwell, [s.n_points for s in c.structures], c.n_plans, int(a.get("sm_count", 148)),
                               int(a.get("dose_kernel", 0)), int(a.get("wide_accum", 0)))
    h = g.gmco_create(c.D, c.structures, c.rx, options(a, c))
    try:
        out = g.gmco_evaluate(h, T, c.weights, want_dose=True, want_grad=True, host=True)
    finally:
        g.gmco_destroy(h)
    return report(E, errors=eval_errors(out, ref), schedule={k: int(v) for k, v in sched.items()},
                  digest=digest(out["dose"], out["F"], out["grad_x"]),
                  # per tensor kernel that ran: [bytes landed in shared memory by TMA, bytes of it read by MMA operands, tensor-pipe cycles x SMs]
                  traffic={k: [int(E.emu_traffic(k.encode(), w)) for w in range(3)]
                           for k in ("k_dose_tc_pair<4, 6>", "k_dose_tc_pair<0, 0>", "k_dose_tc<true>", "k_grad_tc<16>", "k_grad_tc_pair<16>") if E.emu_traffic(k.encode(), 2)},
                  kernels={k: int(E.emu_counter(k.encode())) for k in ("k_dose_tc<true>", "k_dose_tc<false>", "k_dose_tc<false, true>",
                                                                       "k_dose_tc_pair<4, 6>", "k_dose_tc_pair<0, 0>", "k_grad_tc<16>", "k_grad_tc_pair<16>", "k_simt_dose", "k_simt_grad")})


def sc_optimize(g, E, a):
    """gmco_optimize + gmco_result (the device-side WHILE loop, or host-driven rounds in profiling mode) against the oracle's
    optimisation of the same plans: final objective, DVH indices, iteration counts, exit statuses."""
    c = custom_case(a)
    eps = float(a.get("eps", 0.0))
    ref = oracle.optimize(c.D, c.structures, c.rx, c.T0, c.weights, m=c.m, iters=c.iters, eps=eps)
    h = g.gmco_create(c.D, c.structures, c.rx, options(a, c))
    try:
        if a.get("profile"):
            g.gmco_set_profiling(h, True)
        executed0 = int(E.emu_counter(b"executed"))
        g.gmco_optimize(h, c.T0, c.weights, c.iters)
        out = g.gmco_result(h, host=True)
        executed = int(E.emu_counter(b"executed")) - executed0       # kernels that really ran, graph replays included
        st = g.gmco_get_stats(h)
    finally:
        g.gmco_destroy(h)
    rel_f = np.abs(out["objective"] - ref["F"]) / np.maximum(ref["F"], np.finfo(np.float64).tiny)     # F = 0 exactly on both sides: 0
    dvh_pp = np.abs(out["dvh"] - ref["dvh"])
    same_it = out["iters_done"] == ref["iters_done"]
    return report(E, rel_F_max=float(rel_f.max()), rel_F_median=float(np.median(rel_f)), rel_F_p99=float(np.quantile(rel_f, 0.99)),
                  rel_F_over_1e3=int((rel_f > 1e-3).sum()), rel_F_same_iters_max=float(rel_f[same_it].max()) if same_it.any() else None,
                  dvh_pp_max=float(dvh_pp.max()), iters_gpu=out["iters_done"].tolist(), iters_ref=np.asarray(ref["iters_done"]).tolist(),
                  status_gpu=out["plan_status"].tolist(), status_ref=np.asarray(ref["status"]).tolist(),
                  rounds=int(st["rounds"]), launches=int(st["kernel_launches"]), executed=executed, dose_kernel=int(st["dose_kernel"]),
                  digest=digest(out["T"], out["objective"], out["dvh"]),
                  ls_launches=int(E.emu_counter(b"k_ls_pick")), step_launches=int(E.emu_counter(b"k_step")),
                  grad_pair_launches=int(E.emu_counter(b"k_grad_tc_pair")))


def sc_fault(g, E, a):
    """Fault injection: the n-th TMA completion (or tcgen05.commit) after the handle's creation is lost.  The kernels must
    run into their bounded waits, leave through the normal teardown, and the ABI must report GMCO_E_CUDA -- no hang."""
    c = custom_case(a)
    T = np.repeat(c.T0[None], c.n_plans, axis=0)
    h = g.gmco_create(c.D, c.structures, c.rx, options(a, c))
    err, code = "", 0
    t0 = time.time()
    try:
        E.emu_set(a["drop"].encode(), int(a["nth"]))
        try:
            if a.get("via", "evaluate") == "evaluate":
                g.gmco_evaluate(h, T, c.weights, want_dose=False, want_grad=True, host=True)
            else:
                g.gmco_optimize(h, c.T0, c.weights, int(a.get("iters", 3)))
                g.gmco_result(h, host=True)
        except b.GmcoError as ex:
            err, code = str(ex), ex.code
        E.emu_set(a["drop"].encode(), -1)
        # the handle recovers: the same call succeeds once the fault is gone
        after = None
        if not a.get("no_recovery"):
            out = g.gmco_evaluate(h, T, c.weights, want_dose=True, want_grad=True, host=True)
            after = eval_errors(out, oracle.evaluate(c.D, c.structures, T, c.weights))
    finally:
        g.gmco_destroy(h)
    return report(E, error=err, code=code, seconds=time.time() - t0, errors_after=after)


def sc_fault_sweep(g, E, a):
    """Every one of `count` consecutive TMA completions (or commits) of an evaluation lost in turn.  Each run must end
    either in GMCO_E_CUDA or -- where the lost completion is one nobody waits for -- in a correct result; never in a hang."""
    c = custom_case(a)
    T = np.repeat(c.T0[None], c.n_plans, axis=0)
    ref = oracle.evaluate(c.D, c.structures, T, c.weights)
    h = g.gmco_create(c.D, c.structures, c.rx, options(a, c))
    contained = harmless = wrong = 0
    sites = {}
    try:
        first = int(a.get("first", 0))
        for nth in range(first, first + int(a["count"]) * int(a.get("stride", 1)), int(a.get("stride", 1))):
            E.emu_set(a["drop"].encode(), nth)
            try:
                out = g.gmco_evaluate(h, T, c.weights, want_dose=True, want_grad=True, host=True)
                if max(eval_errors(out, ref).values()) < 1e-4:
                    harmless += 1
                else:
                    wrong += 1
            except b.GmcoError as ex:
                contained += 1
                key = str(ex).split("did not complete in ")[-1].split(", block")[0]
                sites[key] = sites.get(key, 0) + 1
            E.emu_set(a["drop"].encode(), -1)
        out = g.gmco_evaluate(h, T, c.weights, want_dose=True, want_grad=True, host=True)
    finally:
        g.gmco_destroy(h)
    return report(E, contained=contained, harmless=harmless, wrong=wrong, sites=sites, errors_after=eval_errors(out, ref))


def sc_sa(g, E, a):
    """gSA chains on the fp64 route: the whole trajectory must equal the oracle's (acceptance counts, dwell times)."""
    c = custom_case(a)
    K, steps = c.n_plans, int(a.get("steps", 300))
    jdx, z, u = gc.sa_draws(c.n_dwell, K, steps, seed=5)
    tau = float(c.T0[0])
    h = g.gmco_create(c.D, c.structures, c.rx, options(a, c))
    try:
        out = g.gmco_sa_run(h, c.T0, c.weights, jdx, z, u, tau, precision=int(a.get("sa_precision", 0)), host=True)
    finally:
        g.gmco_destroy(h)
    acc_ref, t_err, f_err = [], 0.0, 0.0
    for k in range(K):
        r = oracle.sa_chain(c.D, c.structures, c.weights[k], c.T0, tau, jdx[k], z[k], u[k])
        acc_ref.append(int(r["n_accepted"]))
        t_err = max(t_err, float(np.abs(out["T"][k] - r["t"]).max()))
        f_err = max(f_err, float(abs(out["objective"][k] - r["F"]) / r["F"]))
    return report(E, accepted_gpu=out["n_accepted"].tolist(), accepted_ref=acc_ref, T_abs_err=t_err, F_rel_err=f_err)


def sc_exact(g, E, a):
    """Index check with exact arithmetic: D holds small integers (exact in tf32), plan k dwells for exactly 1 s at ONE
    position a_k, so dose[i, k] must equal D[i, a_k] to the last bit on every route -- any slip in a TMA coordinate, a
    swizzle, a descriptor or an accumulator column gives a different integer."""
    c = custom_case(a)
    rng = np.random.Generator(np.random.PCG64(99))
    D = rng.integers(1, 1000, size=c.D.shape).astype(np.float32)
    K, A = c.n_plans, c.n_dwell
    pos = (np.arange(K) * 7 + 3) % A
    T = np.zeros((K, A), np.float32)
    T[np.arange(K), pos] = 1.0
    h = g.gmco_create(D, c.structures, c.rx, options(a, c))
    try:
        out = g.gmco_evaluate(h, T, c.weights, want_dose=True, want_grad=False, host=True)
    finally:
        g.gmco_destroy(h)
    return report(E, exact=bool(np.array_equal(out["dose"], D[:, pos])), mismatches=int((out["dose"] != D[:, pos]).sum()))


def sc_smoke(g, E, a):
    """The call sequence of __graft_entry__.smoke() (same cases, same arguments, same bars), on the emulation."""
    c = gc.make_case("C1")
    ref = oracle.optimize(c.D, c.structures, c.rx, c.T0, c.weights, m=c.m, iters=c.iters)
    legs = {}
    for prec, name in ((b.GMCO_PREC_TF32X3, "tf32x3"), (b.GMCO_PREC_SIMT_FP32, "simt_fp32")):
        h = g.gmco_create(c.D, c.structures, c.rx, b.make_options(m=c.m, precision=prec))
        try:
            ev = g.gmco_evaluate(h, c.T0, c.weights, want_dose=True, host=True)       # 1-D T0: broadcast to all plans
            g.gmco_optimize(h, c.T0, c.weights, c.iters)
            out = g.gmco_result(h, host=True)
        finally:
            g.gmco_destroy(h)
        ref_ev = oracle.evaluate(c.D, c.structures, c.T0, c.weights)
        legs[name] = dict(dose=float(np.abs(ev["dose"] / ref_ev["dose"] - 1).max()), F=float(np.abs(out["objective"] / ref["F"] - 1).max()),
                          dvh_pp=float(np.abs(out["dvh"] - ref["dvh"]).max()))
    c2 = gc.make_case("C1", n_plans=256)
    T = np.repeat(c2.T0[None], 256, axis=0) * np.linspace(0.7, 1.3, 256)[:, None].astype(np.float32)
    h = g.gmco_create(c2.D, c2.structures, c2.rx)
    try:
        ev = g.gmco_evaluate(h, T, c2.weights, want_dose=True, host=True)
    finally:
        g.gmco_destroy(h)
    ref_ev = oracle.evaluate(c2.D, c2.structures, T, c2.weights)
    legs["pair_256"] = dict(dose=float(np.abs(ev["dose"] / ref_ev["dose"] - 1).max()), F=float(np.abs(ev["F"] / ref_ev["F"] - 1).max()),
                            pair_kernel_ran=int(E.emu_counter(b"k_dose_tc_pair")))
    h = g.gmco_create(c.D, c.structures, c.rx)
    try:
        jdx, z, u = gc.sa_draws(c.n_dwell, c.n_plans, 2000, seed=5)
        sa = g.gmco_sa_run(h, c.T0, c.weights, jdx, z, u, float(c.T0[0]), host=True)
    finally:
        g.gmco_destroy(h)
    r = oracle.sa_chain(c.D, c.structures, c.weights[0], c.T0, float(c.T0[0]), jdx[0], z[0], u[0])
    legs["gsa"] = dict(accepted=int(sa["n_accepted"][0]), accepted_ref=int(r["n_accepted"]), F=float(abs(sa["objective"][0] / r["F"] - 1)))
    return report(E, legs=legs)


def sc_pool(g, E, a):
    """Pareto filter and plan selection (comparisons only: bit-exact) and the dose-rate matrix (one fp32 ulp)."""
    rng = np.random.Generator(np.random.PCG64(11))
    K, M = int(a.get("K", 300)), 5
    obj = rng.random((K, M)).astype(np.float32)
    obj[rng.integers(0, K, 20)] = obj[rng.integers(0, K, 20)]          # exact duplicates
    c = custom_case(a)
    h = g.gmco_create(c.D, c.structures, c.rx, options(a, c))
    try:
        pf = g.gmco_pareto_front(h, obj)
        dvh = np.stack([rng.uniform(80, 100, K), rng.uniform(100, 125, K), rng.uniform(0, 3, K), rng.uniform(0, 3, K)], axis=1).astype(np.float32)
        crit = [(0, +1, 90.0, 95.0, 0), (1, -1, 118.0, 115.0, 1), (2, -1, 1.5, 1.0, 2), (3, -1, 1.5, 1.0, 2)]
        sel = g.gmco_select_plan(h, dvh, crit)
    finally:
        g.gmco_destroy(h)
    ref_pf = oracle.pareto_front(obj)
    ref_sel, ref_cls, ref_cnt = oracle.select_plan(dvh, crit)
    D = g.gmco_dose_rate_matrix(c.points, c.dwell, gc.G_COEF, gc.SK_LAMBDA, gc.R_FLOOR_CM, host=True)
    Dref = oracle.dose_rate_matrix(c.points, c.dwell, gc.G_COEF, gc.SK_LAMBDA, gc.R_FLOOR_CM)
    ulp = np.abs(D.view(np.int32).astype(np.int64) - Dref.view(np.int32).astype(np.int64))
    return report(E, pareto_equal=bool(np.array_equal(pf["nondominated"], ref_pf)), n_nondominated=int(pf["n_nondominated"]),
                  selected=int(sel["selected"]), selected_ref=int(ref_sel), classes_equal=bool(np.array_equal(sel["plan_class"], ref_cls)),
                  class_counts_equal=bool(np.array_equal(sel["class_counts"], ref_cnt)),
                  dose_rate=dict(max_ulp=int(ulp.max()), exact_fraction=float((ulp == 0).mean())))


SCENARIOS = {"exact": sc_exact, "smoke": sc_smoke, "fault_sweep": sc_fault_sweep, "evaluate": sc_evaluate, "optimize": sc_optimize, "fault": sc_fault, "sa": sc_sa, "pool": sc_pool}


def main():
    a = json.loads(sys.argv[1])
    lib = Path(a.get("lib", ROOT / "tests" / "emu" / "_build" / "libgmco_emu.so"))
    g, E = load(lib)
    configure(E, a)
    t0 = time.time()
    try:
        out = SCENARIOS[a["scenario"]](g, E, a)
    except b.GmcoError as ex:                  # a scenario that does not expect an error: report it instead of dying
        out = report(E, error=str(ex), code=ex.code)
    out["seconds"] = out.get("seconds", time.time() - t0)
    if a.get("times"):
        E.emu_print_times()
    print("EMU_RESULT " + json.dumps(out))


if __name__ == "__main__":
    main()
