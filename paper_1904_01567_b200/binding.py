"""ctypes binding of libgmco.so: same names as include/gmco.h, marshalling only."""
from __future__ import annotations

import ctypes as C
from pathlib import Path

import numpy as np

_PKG = Path(__file__).resolve().parent
GMCO_PREC_TF32X3, GMCO_PREC_SIMT_FP32 = 0, 1
GMCO_MAX_STRUCTS = 8
GMCO_SA_FP64, GMCO_SA_FP32 = 0, 1


class GmcoError(RuntimeError):
    def __init__(self, code, msg):
        super().__init__(f"libgmco error {code}: {msg}")
        self.code = code


class _Structure(C.Structure):
    _fields_ = [("n_points", C.c_int32), ("d_lo", C.c_float), ("d_hi", C.c_float), ("w_lo", C.c_float),
                ("w_hi", C.c_float), ("dvh_kind", C.c_int32), ("dvh_level", C.c_float)]


class Options(C.Structure):
    _fields_ = [("m", C.c_int32), ("eps", C.c_float), ("c1", C.c_float), ("max_trials", C.c_int32),
                ("precision", C.c_int32), ("eps_f", C.c_float), ("compaction", C.c_int32), ("dose_kernel", C.c_int32),
                ("wide_accum", C.c_int32), ("line_search", C.c_int32)]


class Criterion(C.Structure):
    _fields_ = [("structure", C.c_int32), ("sense", C.c_int32), ("limit_rtog", C.c_float),
                ("limit_rtog_plus", C.c_float), ("role", C.c_int32)]


class Stats(C.Structure):
    _fields_ = [("device_bytes", C.c_int64), ("rounds", C.c_int32), ("kernel_launches", C.c_int32),
                ("plans_iters", C.c_int32), ("plans_converged", C.c_int32), ("plans_stalled", C.c_int32),
                ("eval_launches", C.c_int32), ("eval_ms", C.c_float), ("eval_plans", C.c_int32),
                ("dose_ms", C.c_float), ("grad_ms", C.c_float), ("step_ms", C.c_float), ("dose_kernel", C.c_int32)]


class TcInfo(C.Structure):
    _fields_ = [(n, C.c_int32) for n in (
        "ok", "a_pad", "n_pad", "n_alloc", "k_pad", "n_tiles", "segs", "n_chunks", "n_slabs", "compact_cap", "dose_kernel",
        "dose_threads", "dose_stages", "dose_stage_bytes", "dose_smem_bytes", "dose_smem_end", "dose_scr_slot", "dose_tmem_cols",
        "dose_tmem_groups", "dose_n_main",
        "grad_threads", "grad_ps", "grad_stages", "grad_stage_bytes", "grad_smem_bytes", "grad_smem_end", "grad_staging_bytes",
        "grad_tmem_cols", "smem_limit", "tmem_limit", "grad_pair")]

DOSE_KERNEL_NAMES = {-1: "k_simt_dose", 0: "k_dose_tc<resident>", 1: "k_dose_tc<streamed>", 2: "k_dose_tc_pair<4,6>",
                     3: "k_dose_tc_pair<0,0>"}


def lib_path() -> Path:
    return _PKG / "libgmco.so"


_lib = None


def lib():
    """Load libgmco.so.  Raises (never falls back) when it is missing: build it with
    ``python -m paper_1904_01567_b200.build`` or ``__graft_entry__.build()``."""
    global _lib
    if _lib is None:
        p = lib_path()
        if not p.exists():
            raise ImportError(f"{p} is missing: run `python paper_1904_01567_b200/build.py` (needs nvcc). "
                              "There is no CPU fallback.")
        L = C.CDLL(str(p))
        vp, i32, i64, fp = C.c_void_p, C.c_int32, C.c_int64, C.c_void_p
        L.gmco_version.restype = C.c_int
        L.gmco_default_options.argtypes = [C.POINTER(Options)]
        L.gmco_default_options.restype = None
        L.gmco_create.argtypes = [C.POINTER(vp), fp, i64, i64, i64, C.POINTER(_Structure), i32, C.c_float,
                                  C.POINTER(Options), vp]
        L.gmco_optimize.argtypes = [vp, fp, i32, fp, i32, i32, vp]
        L.gmco_result.argtypes = [vp, fp, fp, fp, fp, vp, vp]
        L.gmco_evaluate.argtypes = [vp, fp, i32, fp, i32, fp, fp, fp, vp]
        L.gmco_sa_run.argtypes = [vp, fp, i32, fp, i32, i64, vp, vp, vp, i32, C.c_double, C.c_double, C.c_double,
                                  i32, vp, vp, vp, vp]
        L.gmco_dose_rate_matrix.argtypes = [fp, i64, fp, i64, C.POINTER(C.c_double), i32, C.c_double, C.c_double, fp, i64, vp]
        L.gmco_select_plan.argtypes = [vp, fp, i32, C.POINTER(Criterion), i32, vp, vp, vp, vp]
        L.gmco_pareto_front.argtypes = [vp, fp, i32, i32, vp, vp, vp]
        L.gmco_get_stats.argtypes = [vp, C.POINTER(Stats)]
        L.gmco_tc_schedule.argtypes = [i64, C.POINTER(i32), i32, i32, i32, i32, i32, C.POINTER(TcInfo)]
        L.gmco_set_profiling.argtypes = [vp, i32]
        L.gmco_destroy.argtypes = [vp]
        L.gmco_destroy.restype = None
        L.gmco_last_error.argtypes = [vp]
        L.gmco_last_error.restype = C.c_char_p
        _lib = L
    return _lib


def gmco_version() -> int:
    return int(lib().gmco_version())


class Handle:
    def __init__(self, ptr, n_points, n_dwell, n_structs):
        self.ptr, self.n_points, self.n_dwell, self.n_structs = ptr, n_points, n_dwell, n_structs
        self.K = 0
        self._keep = []          # inputs that must outlive the enqueued work


def _check(rc, h=None):
    if rc != 0:
        msg = lib().gmco_last_error(h.ptr if h is not None else None)
        raise GmcoError(rc, msg.decode() if msg else "")


def _ptr(a):
    """Raw address of a torch tensor (any device) or numpy array; None -> NULL."""
    if a is None:
        return None
    if isinstance(a, np.ndarray):
        assert a.flags["C_CONTIGUOUS"]
        return a.ctypes.data
    assert a.is_contiguous()
    return a.data_ptr()


def _f32(a):
    if isinstance(a, np.ndarray):
        return np.ascontiguousarray(a, dtype=np.float32)
    import torch
    return a.to(torch.float32).contiguous()


def _stream(stream):
    if stream is None:
        import torch
        if torch.cuda.is_available():
            return torch.cuda.current_stream().cuda_stream
        return None
    return getattr(stream, "cuda_stream", stream)


def make_options(m=10, eps=0.0, c1=1e-4, max_trials=20, precision=GMCO_PREC_TF32X3, eps_f=None, compaction=None,
                 dose_kernel=None, wide_accum=None, line_search=None) -> Options:
    o = Options()
    lib().gmco_default_options(C.byref(o))
    o.m, o.eps, o.c1, o.max_trials, o.precision = m, eps, c1, max_trials, precision
    if eps_f is not None:
        o.eps_f = eps_f
    if compaction is not None:
        o.compaction = int(compaction)
    if dose_kernel is not None:
        o.dose_kernel = int(dose_kernel)
    if wide_accum is not None:
        o.wide_accum = int(wide_accum)
    if line_search is not None:
        o.line_search = int(line_search)
    return o


def gmco_create(D, structures, rx, options: Options | None = None, stream=None) -> Handle:
    """D: [n_points, n_dwell] fp32 tensor/array (host or device); structures: objects with the
    fields of gmco_structure (e.g. gmco_cases.Structure)."""
    D = _f32(D)
    n_points, n_dwell = int(D.shape[0]), int(D.shape[1])
    st = (_Structure * len(structures))()
    for i, s in enumerate(structures):
        st[i] = _Structure(int(s.n_points), float(s.d_lo), float(s.d_hi), float(s.w_lo), float(s.w_hi),
                           int(s.dvh_kind), float(s.dvh_level))
    out = C.c_void_p()
    rc = lib().gmco_create(C.byref(out), _ptr(D), n_points, n_dwell, n_dwell, st, len(structures), float(rx),
                           C.byref(options) if options is not None else None, _stream(stream))
    _check(rc)
    h = Handle(out, n_points, n_dwell, len(structures))
    h._keep.append(D)
    return h


def gmco_optimize(h: Handle, T0, weights, iters: int, stream=None) -> None:
    T0, weights = _f32(T0), _f32(weights)
    K = int(weights.shape[0]) if weights.ndim == 3 else int(weights.numel() if hasattr(weights, "numel") else weights.size) // (2 * h.n_structs)
    bc = 1 if T0.ndim == 1 else 0
    h._keep = h._keep[:1] + [T0, weights]
    h.K = K
    _check(lib().gmco_optimize(h.ptr, _ptr(T0), bc, _ptr(weights), K, int(iters), _stream(stream)), h)


def gmco_result(h: Handle, host: bool = False, want_terms: bool = True) -> dict:
    """Returns dict(T, objective, dvh, objective_terms, iters_done, plan_status) as device tensors
    (or numpy arrays when host=True)."""
    K, A, S = h.K, h.n_dwell, h.n_structs
    if host:
        T = np.empty((K, A), np.float32); F = np.empty(K, np.float32); dvh = np.empty((K, S), np.float32)
        terms = np.empty((K, S, 2), np.float32) if want_terms else None
        it = np.empty(K, np.int32); stt = np.empty(K, np.int32)
    else:
        import torch
        dev = torch.device("cuda")
        T = torch.empty((K, A), dtype=torch.float32, device=dev); F = torch.empty(K, dtype=torch.float32, device=dev)
        dvh = torch.empty((K, S), dtype=torch.float32, device=dev)
        terms = torch.empty((K, S, 2), dtype=torch.float32, device=dev) if want_terms else None
        it = torch.empty(K, dtype=torch.int32, device=dev); stt = torch.empty(K, dtype=torch.int32, device=dev)
    _check(lib().gmco_result(h.ptr, _ptr(T), _ptr(F), _ptr(dvh), _ptr(terms), _ptr(it), _ptr(stt)), h)
    return dict(T=T, objective=F, dvh=dvh, objective_terms=terms, iters_done=it, plan_status=stt)


def gmco_evaluate(h: Handle, T, weights, want_dose=False, want_grad=True, host: bool = False, stream=None) -> dict:
    T, weights = _f32(T), _f32(weights)
    K = int(weights.shape[0])
    bc = 1 if T.ndim == 1 else 0
    N, A = h.n_points, h.n_dwell
    if host:
        dose = np.empty((N, K), np.float32) if want_dose else None
        F = np.empty(K, np.float32); g = np.empty((K, A), np.float32) if want_grad else None
    else:
        import torch
        dev = torch.device("cuda")
        dose = torch.empty((N, K), dtype=torch.float32, device=dev) if want_dose else None
        F = torch.empty(K, dtype=torch.float32, device=dev)
        g = torch.empty((K, A), dtype=torch.float32, device=dev) if want_grad else None
    h._keep = h._keep[:1] + [T, weights]
    h.K = K
    _check(lib().gmco_evaluate(h.ptr, _ptr(T), bc, _ptr(weights), K, _ptr(dose), _ptr(F), _ptr(g), _stream(stream)), h)
    return dict(dose=dose, F=F, grad_x=g)


def gmco_sa_run(h: Handle, T0, weights, jdx, z, u, tau: float, temp0: float = 1.0, cooling: float = 0.995,
                precision: int = GMCO_SA_FP64, host: bool = False, stream=None) -> dict:
    """K simulated-annealing chains (include/gmco.h gmco_sa_run).  jdx int32, z / u fp64, each [K][steps] or [steps]
    (shared by all chains).  Returns dict(T [K][A] fp64, objective [K] fp64, n_accepted [K] int64)."""
    T0, weights = _f32(T0), _f32(weights)
    K = int(weights.shape[0])
    bc = 1 if T0.ndim == 1 else 0
    if isinstance(jdx, np.ndarray):
        jdx = np.ascontiguousarray(jdx, dtype=np.int32)
        z = np.ascontiguousarray(z, dtype=np.float64); u = np.ascontiguousarray(u, dtype=np.float64)
    else:
        import torch
        jdx = jdx.to(torch.int32).contiguous(); z = z.to(torch.float64).contiguous(); u = u.to(torch.float64).contiguous()
    dbc = 1 if jdx.ndim == 1 else 0
    steps = int(jdx.shape[-1])
    assert tuple(z.shape) == tuple(jdx.shape) == tuple(u.shape) and (dbc or int(jdx.shape[0]) == K)
    A = h.n_dwell
    if host:
        T = np.empty((K, A), np.float64); F = np.empty(K, np.float64); na = np.empty(K, np.int64)
    else:
        import torch
        dev = torch.device("cuda")
        T = torch.empty((K, A), dtype=torch.float64, device=dev); F = torch.empty(K, dtype=torch.float64, device=dev)
        na = torch.empty(K, dtype=torch.int64, device=dev)
    _check(lib().gmco_sa_run(h.ptr, _ptr(T0), bc, _ptr(weights), K, steps, _ptr(jdx), _ptr(z), _ptr(u), dbc,
                             float(tau), float(temp0), float(cooling), int(precision), _ptr(T), _ptr(F), _ptr(na),
                             _stream(stream)), h)
    return dict(T=T, objective=F, n_accepted=na)


def gmco_dose_rate_matrix(points_mm, dwell_mm, g_coef, sk_lambda: float, r_floor_cm: float, host: bool = False, stream=None):
    """Step (i): D [N, A] fp32 (device tensor, or numpy when host=True) from coordinates in millimetres."""
    p, q = _f32(points_mm), _f32(dwell_mm)
    N, A = int(p.shape[0]), int(q.shape[0])
    coef = (C.c_double * len(g_coef))(*[float(c) for c in g_coef])
    if host:
        D = np.empty((N, A), np.float32)
    else:
        import torch
        D = torch.empty((N, A), dtype=torch.float32, device="cuda")
    _check(lib().gmco_dose_rate_matrix(_ptr(p), N, _ptr(q), A, coef, len(g_coef), float(sk_lambda), float(r_floor_cm),
                                       _ptr(D), A, _stream(stream)))
    return D


def gmco_select_plan(h: Handle, dvh, criteria, stream=None) -> dict:
    """criteria: sequence of (structure, sense, limit_rtog, limit_rtog_plus, role).  Returns dict(selected, plan_class
    [K] int32 numpy, class_counts [3])."""
    dvh = _f32(dvh)
    K = int(dvh.shape[0])
    arr = (Criterion * len(criteria))(*[Criterion(int(c[0]), int(c[1]), float(c[2]), float(c[3]), int(c[4])) for c in criteria])
    cls = np.empty(K, np.int32); sel = np.empty(1, np.int32); cnt = np.empty(3, np.int32)
    _check(lib().gmco_select_plan(h.ptr, _ptr(dvh), K, arr, len(criteria), _ptr(cls), _ptr(sel), _ptr(cnt),
                                  _stream(stream)), h)
    return dict(selected=int(sel[0]), plan_class=cls, class_counts=cnt)


def gmco_pareto_front(h: Handle, objectives, stream=None) -> dict:
    """objectives [K][M] (every column minimised).  Returns dict(nondominated [K] bool numpy, n_nondominated)."""
    obj = _f32(objectives)
    K = int(obj.shape[0]); M = int(np.prod(obj.shape[1:])) if K else int(np.prod(obj.shape[1:]) or 1)
    mask = np.empty(K, np.uint8); n = np.empty(1, np.int32)
    _check(lib().gmco_pareto_front(h.ptr, _ptr(obj), K, M, _ptr(mask), _ptr(n), _stream(stream)), h)
    return dict(nondominated=mask.astype(bool), n_nondominated=int(n[0]))


def gmco_get_stats(h: Handle) -> dict:
    s = Stats()
    _check(lib().gmco_get_stats(h.ptr, C.byref(s)), h)
    return {k: getattr(s, k) for k, _ in Stats._fields_ if k != "reserved"}


def gmco_tc_schedule(n_dwell: int, struct_points, K: int, num_sms: int = 148, dose_kernel: int = 0, wide_accum: int = 0) -> dict:
    """Launch schedule and on-chip layout of the tensor route for a shape (host arithmetic; needs no GPU)."""
    pts = (C.c_int32 * len(struct_points))(*[int(v) for v in struct_points])
    info = TcInfo()
    _check(lib().gmco_tc_schedule(int(n_dwell), pts, len(struct_points), int(K), int(num_sms), int(dose_kernel), int(wide_accum),
                                  C.byref(info)))
    return {k: getattr(info, k) for k, _ in TcInfo._fields_}


def gmco_set_profiling(h: Handle, enable: bool) -> None:
    _check(lib().gmco_set_profiling(h.ptr, 1 if enable else 0), h)


def gmco_destroy(h: Handle) -> None:
    if h is not None and h.ptr:
        lib().gmco_destroy(h.ptr)
        h.ptr = None
        h._keep = []
