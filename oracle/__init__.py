"""ctypes front end of the fp64 CPU oracle (``oracle/gmco_oracle.c``).

TEST INFRASTRUCTURE, NOT THE PRODUCT: only ``tests/``, ``__graft_entry__.smoke()``
and ``bench.py``'s ``cpu_baseline`` / ``--impl reference`` legs may import this
package.  It imports nothing from ``paper_1904_01567_b200`` and shares no code with
the CUDA path; the only shared module is the arithmetic-free input generator
``gmco_cases``.  This file does argument marshalling only -- every formula lives in
the C file, next to the PAPER.md passage it restates.
"""
from __future__ import annotations

import ctypes as C
import os
import subprocess
from pathlib import Path

import numpy as np

_HERE = Path(__file__).resolve().parent
_SRC = _HERE / "gmco_oracle.c"
_LIB = _HERE / "_build" / "libgmco_oracle.so"


def build(force: bool = False) -> Path:
    """Compile the C oracle with gcc (plain -O2, OpenMP over plans)."""
    if force or not _LIB.exists() or _LIB.stat().st_mtime < _SRC.stat().st_mtime:
        _LIB.parent.mkdir(exist_ok=True)
        tmp = _LIB.with_suffix(f".{os.getpid()}.tmp")
        subprocess.run(["gcc", "-O2", "-std=c11", "-fopenmp", "-fPIC", "-shared", "-Wall",
                        "-o", str(tmp), str(_SRC), "-lm"], check=True)
        os.replace(tmp, _LIB)
    return _LIB


class OrcStruct(C.Structure):
    _fields_ = [("n_points", C.c_int32), ("d_lo", C.c_double), ("d_hi", C.c_double),
                ("w_lo", C.c_double), ("w_hi", C.c_double), ("dvh_kind", C.c_int32),
                ("dvh_level", C.c_double)]


class LbfgsOpt(C.Structure):
    _fields_ = [("m", C.c_int32), ("iters", C.c_int32), ("eps", C.c_double), ("c1", C.c_double),
                ("max_trials", C.c_int32), ("eps_f", C.c_double)]


class LbfgsStat(C.Structure):
    _fields_ = [("iters_done", C.c_int32), ("status", C.c_int32), ("n_evals", C.c_int32),
                ("n_backtracks", C.c_int32), ("n_skipped", C.c_int32), ("n_approx", C.c_int32),
                ("n_bt_iters", C.c_int32), ("max_bt_iter", C.c_int32)]


EPS_F = 1e-6   # default objective-noise allowance of the approximate line-search test (reading A5b)

FG_FN = C.CFUNCTYPE(C.c_double, C.POINTER(C.c_double), C.POINTER(C.c_double), C.c_void_p)

_lib = None


def lib():
    global _lib
    if _lib is None:
        _lib = C.CDLL(str(build()))
        _lib.orc_eval_plan.restype = C.c_double
        _lib.orc_num_threads.restype = C.c_int
    return _lib


def num_threads() -> int:
    return int(lib().orc_num_threads())


def _structs(structures):
    arr = (OrcStruct * len(structures))()
    for i, s in enumerate(structures):
        arr[i] = OrcStruct(int(s.n_points), float(s.d_lo), float(s.d_hi), float(s.w_lo),
                           float(s.w_hi), int(s.dvh_kind), float(s.dvh_level))
    return arr


def _f32(a):
    return np.ascontiguousarray(a, dtype=np.float32)


def _p(a, ty=C.c_double):
    return None if a is None else a.ctypes.data_as(C.POINTER(ty))


def eval_plan(D, structures, w, x):
    """One plan at dwell WEIGHTS x (fp64).  Returns dict(F, dose, Fterm, r, G, g)."""
    D = _f32(D); N, A = D.shape; S = len(structures)
    w = _f32(w).reshape(S, 2); x = np.ascontiguousarray(x, dtype=np.float64)
    dose = np.empty(N); Ft = np.empty((S, 2)); r = np.empty(N); G = np.empty(A); g = np.empty(A)
    F = lib().orc_eval_plan(_p(D, C.c_float), C.c_int64(N), C.c_int64(A), _structs(structures),
                            C.c_int32(S), _p(w, C.c_float), _p(x), _p(dose), _p(Ft), _p(r), _p(G), _p(g))
    return dict(F=float(F), dose=dose, Fterm=Ft, r=r, G=G, g=g)


def evaluate(D, structures, T, weights, want_dose=True):
    """Batch evaluation at dwell TIMES T ([K, A] or [A], fp32).  dose is [N, K]."""
    D = _f32(D); N, A = D.shape; S = len(structures)
    weights = _f32(weights).reshape(-1, S, 2); K = weights.shape[0]
    T = _f32(T); bc = 1 if T.ndim == 1 else 0
    dose = np.empty((N, K)) if want_dose else None
    F = np.empty(K); Ft = np.empty((K, S, 2)); gx = np.empty((K, A)); G = np.empty((K, A))
    rc = lib().orc_evaluate(_p(D, C.c_float), C.c_int64(N), C.c_int64(A), _structs(structures),
                            C.c_int32(S), _p(T, C.c_float), C.c_int32(bc), _p(weights, C.c_float),
                            C.c_int32(K), _p(dose), _p(F), _p(Ft), _p(gx), _p(G))
    if rc != 0:
        raise ValueError("orc_evaluate: structure sizes do not add up to N")
    return dict(F=F, dose=dose, Fterm=Ft, grad_x=gx, G=G)


def lbfgs(fg, x0, m=10, iters=100, eps=0.0, c1=1e-4, max_trials=20, eps_f=EPS_F):
    """Generic driver on a Python objective fg(x) -> (F, g); used to PIN the driver."""
    x = np.array(x0, dtype=np.float64); n = x.size

    def _cb(xp, gp, _ctx):
        xv = np.ctypeslib.as_array(xp, shape=(n,))
        F, g = fg(xv.copy())
        np.ctypeslib.as_array(gp, shape=(n,))[:] = g
        return float(F)

    cb = FG_FN(_cb)
    opt = LbfgsOpt(m, iters, eps, c1, max_trials, eps_f); st = LbfgsStat()
    Ff = C.c_double(); hist = np.empty(iters + 1)
    lib().orc_lbfgs(cb, None, C.c_int64(n), _p(x), C.byref(opt), C.byref(Ff), _p(hist), C.byref(st))
    return dict(x=x, F=Ff.value, F_hist=hist, iters_done=st.iters_done, status=st.status,
                n_evals=st.n_evals, n_backtracks=st.n_backtracks, n_skipped=st.n_skipped, n_approx=st.n_approx,
                n_bt_iters=st.n_bt_iters, max_bt_iter=st.max_bt_iter)


def optimize(D, structures, rx, T0, weights, m=10, iters=100, eps=0.0, c1=1e-4, max_trials=20,
             want_hist=False, eps_f=EPS_F):
    """K plans of gL-BFGS from dwell times T0 ([K, A] or [A]).  Returns dict of fp64 arrays."""
    D = _f32(D); N, A = D.shape; S = len(structures)
    weights = _f32(weights).reshape(-1, S, 2); K = weights.shape[0]
    T0 = _f32(T0); bc = 1 if T0.ndim == 1 else 0
    opt = LbfgsOpt(m, iters, eps, c1, max_trials, eps_f)
    T = np.empty((K, A)); F = np.empty(K); dvh = np.empty((K, S)); Ft = np.empty((K, S, 2))
    stats = (LbfgsStat * K)(); hist = np.empty((K, iters + 1)) if want_hist else None
    rc = lib().orc_optimize(_p(D, C.c_float), C.c_int64(N), C.c_int64(A), _structs(structures),
                            C.c_int32(S), C.c_double(rx), _p(T0, C.c_float), C.c_int32(bc),
                            _p(weights, C.c_float), C.c_int32(K), C.byref(opt),
                            _p(T), _p(F), _p(dvh), _p(Ft), stats, _p(hist))
    if rc != 0:
        raise ValueError("orc_optimize: structure sizes do not add up to N")
    return dict(T=T, F=F, dvh=dvh, Fterm=Ft, F_hist=hist,
                iters_done=np.array([s.iters_done for s in stats]),
                status=np.array([s.status for s in stats]),
                n_evals=np.array([s.n_evals for s in stats]),
                n_backtracks=np.array([s.n_backtracks for s in stats]),
                n_skipped=np.array([s.n_skipped for s in stats]),
                n_approx=np.array([s.n_approx for s in stats]),
                n_bt_iters=np.array([s.n_bt_iters for s in stats]),
                max_bt_iter=np.array([s.max_bt_iter for s in stats]))


def dvh(dose, structures, rx):
    dose = np.ascontiguousarray(dose, dtype=np.float64); out = np.empty(len(structures))
    lib().orc_dvh(_p(dose), _structs(structures), C.c_int32(len(structures)), C.c_double(rx), _p(out))
    return out


def sa_chain(D, structures, w, T0, tau, jdx, z, u, temp0=1.0, cooling=0.995, want_dose=False):
    """One simulated-annealing chain; the random draws jdx, z, u are inputs."""
    D = _f32(D); N, A = D.shape; S = len(structures)
    w = _f32(w).reshape(S, 2); T0 = _f32(T0)
    jdx = np.ascontiguousarray(jdx, dtype=np.int32); steps = jdx.size
    z = np.ascontiguousarray(z, dtype=np.float64); u = np.ascontiguousarray(u, dtype=np.float64)
    t = np.empty(A); d = np.empty(N) if want_dose else None; F = C.c_double(); na = C.c_int64()
    lib().orc_sa_chain(_p(D, C.c_float), C.c_int64(N), C.c_int64(A), _structs(structures), C.c_int32(S),
                       _p(w, C.c_float), _p(T0, C.c_float), C.c_double(tau), C.c_int64(steps),
                       _p(jdx, C.c_int32), _p(z), _p(u), C.c_double(temp0), C.c_double(cooling),
                       _p(t), _p(d), C.byref(F), C.byref(na))
    return dict(t=t, dose=d, F=F.value, n_accepted=na.value)


def pareto_front(objectives):
    """Non-dominated plans (a solution is Pareto optimal "if no solution that improves any individual
    objective value without worsening at least one of the other individual objective values exists").
    objectives [K, M], every column minimised.  The definition written out as a double loop: plan a dominates plan b
    if a_m <= b_m for every m and a_m < b_m for at least one m.  Comparisons only, on the fp32 values as given."""
    obj = np.asarray(objectives, dtype=np.float32).reshape(len(objectives), -1)
    K = obj.shape[0]
    nondom = np.ones(K, dtype=bool)
    for b in range(K):
        for a in range(K):
            if np.all(obj[a] <= obj[b]) and np.any(obj[a] < obj[b]):
                nondom[b] = False
                break
    return nondom


def select_plan(dvh, criteria):
    """Plan evaluation and selection (PAPER.md:132-143 criteria; PAPER.md:147-151 selection; A22-A23).
    dvh [K, S]; criteria: sequence of (structure, sense, limit_rtog, limit_rtog_plus, role) with sense +1 ("index >=
    limit") or -1 ("index < limit") and role 0 target / 1 must-hold / 2 organ at risk.
    Returns (selected index or -1, plan_class [K] with 2 = RTOG+, 1 = RTOG, 0 = invalid, class_counts [3]).
    fp32 comparisons; the fallback's sum of the role-2 indices is an fp32 sum in criterion order."""
    dvh = np.asarray(dvh, dtype=np.float32)
    K = dvh.shape[0]
    cls = np.zeros(K, dtype=np.int32)
    target = np.zeros(K, dtype=np.float32); oar = np.zeros(K, dtype=np.float32); core = np.ones(K, dtype=bool)
    for k in range(K):
        rtog = plus = True
        s = np.float32(0.0)
        for (st, sense, lim, lim_plus, role) in criteria:
            v = dvh[k, st]
            ok = (v >= np.float32(lim)) if sense > 0 else (v < np.float32(lim))
            okp = (v >= np.float32(lim_plus)) if sense > 0 else (v < np.float32(lim_plus))
            rtog = rtog and ok
            plus = plus and okp
            if role == 0:
                target[k] = v
            if role != 2:
                core[k] = core[k] and ok
            if role == 2:
                s = np.float32(s + v)
        oar[k] = s
        cls[k] = 2 if (rtog and plus) else (1 if rtog else 0)
    counts = np.array([(cls == 0).sum(), (cls == 1).sum(), (cls == 2).sum()], dtype=np.int32)
    if K == 0:
        return -1, cls, counts

    def argbest(mask, key):                 # highest key, ties to the lowest index
        idx = np.flatnonzero(mask)
        return int(idx[np.argmax(key[idx])]) if idx.size else -1   # np.argmax returns the first maximum

    for mask, key in ((cls == 2, target), (cls >= 1, target), (core, -oar), (np.ones(K, bool), -oar)):
        sel = argbest(mask, key)
        if sel >= 0:
            return sel, cls, counts
    return -1, cls, counts


def dose_rate_matrix(points_mm, dwell_mm, g_coef, sk_lambda, r_floor_cm):
    """Step (i): D [N, A] fp32 from point and dwell coordinates in mm (orc_dose_rate)."""
    p = _f32(points_mm).reshape(-1, 3); q = _f32(dwell_mm).reshape(-1, 3)
    coef = np.ascontiguousarray(g_coef, dtype=np.float64)
    D = np.empty((p.shape[0], q.shape[0]), np.float32)
    rc = lib().orc_dose_rate(_p(p, C.c_float), C.c_int64(p.shape[0]), _p(q, C.c_float), C.c_int64(q.shape[0]),
                             _p(coef), C.c_int32(coef.size), C.c_double(sk_lambda), C.c_double(r_floor_cm),
                             _p(D, C.c_float))
    if rc != 0:
        raise ValueError("orc_dose_rate: bad arguments")
    return D
