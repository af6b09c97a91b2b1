"""The whole tensor route as a numpy MODEL, optimised end to end and held to the oracle at north_star's bar (no GPU).

Pieces: the arithmetic model of tests/test_tc_arithmetic_model.py (tf32 operand split, one truncating fp32 add per K = 8
step, fp32 epilogue with Eq. 2, gradient contraction with its split of R and the fixed-order segment sum) and the round
protocol of tests/test_step_logic_model.py run in fp32 (k_step: two-loop recursion, Armijo / approximate test, history
ring).  C1 (8 plans, 50 iterations, m = 5) and a 12-plan cut of a C2-shaped case go through the model; iteration counts
must equal the fp64 oracle's, final objectives agree within 1e-3 and DVH indices within 0.5 percentage points.
What this shows while no GPU can be used: the PRECISION DESIGN of the route (3xTF32 with a truncating accumulate, fp32
optimiser state, the approximate line-search test) meets the parity bar after a full optimisation.  It is a model
written by hand from the kernels, not the kernels; the -m gpu tests hold the code itself to the same bar."""
import importlib.util
from pathlib import Path

import numpy as np
import pytest

import gmco_cases as gc
import oracle

HERE = Path(__file__).parent


def _load(name):
    spec = importlib.util.spec_from_file_location(name, HERE / f"{name}.py")
    mod = importlib.util.module_from_spec(spec)
    spec.loader.exec_module(mod)
    return mod


arith = _load("test_tc_arithmetic_model")
steps = _load("test_step_logic_model")
f32 = np.float32


class ModelCase:
    """The library's padded row layout (structures padded to 64 rows, dwell columns to 32) and per-row tables."""

    def __init__(self, c):
        self.c, self.A, self.A_pad = c, c.n_dwell, (c.n_dwell + 31) // 32 * 32
        blocks, sid, valid, off = [], [], [], 0
        for si, s in enumerate(c.structures):
            n_pad = (s.n_points + 63) // 64 * 64
            blk = np.zeros((n_pad, self.A_pad), f32); blk[:s.n_points, :self.A] = c.D[off:off + s.n_points]
            blocks.append(blk); sid += [si] * n_pad; valid += [True] * s.n_points + [False] * (n_pad - s.n_points); off += s.n_points
        self.D, self.sid, self.valid = np.concatenate(blocks), np.array(sid), np.array(valid)
        st = c.structures
        self.d_lo = np.array([st[s].d_lo for s in self.sid], f32); self.d_hi = np.array([st[s].d_hi for s in self.sid], f32)
        self.scale_lo = np.array([st[s].w_lo / st[s].n_points for s in self.sid], f32)
        self.scale_hi = np.array([st[s].w_hi / st[s].n_points for s in self.sid], f32)
        self.segs = min(37, self.D.shape[0] // 16)

    def evaluate(self, X, w):
        """X [K, A_pad] fp32 trial points, w [K, S, 2] -> F [K], g [K, A_pad] as the dose kernel, the gradient kernel and
        the head of k_step would form them."""
        T = (X * X).astype(f32)
        d = arith.dose_model(self.D, T, "sep")
        W_lo = (w[:, self.sid, 0] * self.scale_lo[None]).astype(f32); W_hi = (w[:, self.sid, 1] * self.scale_hi[None]).astype(f32)
        lo = np.minimum(d - self.d_lo[None], f32(0)); hi = np.maximum(d - self.d_hi[None], f32(0))
        u, v = (W_lo * lo).astype(f32), (W_hi * hi).astype(f32)
        f = ((u * lo).astype(f32) + (v * hi).astype(f32)).astype(f32)
        f[:, ~self.valid] = 0
        F = f.sum(axis=1, dtype=f32)
        Rh = (u + v).astype(f32); Rh[:, ~self.valid] = 0
        G = arith.grad_model(self.D, Rh, self.segs, self.A_pad <= 256)
        return F, (f32(4) * X * G).astype(f32)

    def dose(self, X):
        d = arith.dose_model(self.D, (X * X).astype(f32), "sep")
        starts = np.cumsum([0] + [((s.n_points + 63) // 64) * 64 for s in self.c.structures[:-1]])
        return np.concatenate([d[:, o:o + s.n_points] for o, s in zip(starts, self.c.structures)], axis=1)


def optimise_model(c, iters):
    mc = ModelCase(c)
    K = c.n_plans
    w = c.weights.astype(f32)
    x0 = np.zeros(mc.A_pad, f32); x0[:mc.A] = np.sqrt(c.T0.astype(f32))
    states = []
    for k in range(K):
        s = steps.PlanState(x0.astype(np.float64), c.m)
        for name in ("x", "xt", "g", "p", "S", "Y", "rho", "gam"):
            setattr(s, name, getattr(s, name).astype(f32))
        states.append(s)
    rounds = 0
    while any(s.status == steps.RUNNING for s in states) and rounds < 1 + iters * 21:
        run = [k for k in range(K) if states[k].status == steps.RUNNING]
        X = np.stack([states[k].xt for k in run]).astype(f32)
        F, g = mc.evaluate(X, w[run])
        for j, k in enumerate(run):
            s = states[k]
            steps.k_step_model(s, f32(F[j]), g[j], c.m, iters, 20, f32(1e-4), f32(0.0), f32(oracle.EPS_F))
            for name in ("x", "xt", "g", "p"):                       # the kernel keeps its state in fp32
                setattr(s, name, getattr(s, name).astype(f32))
            s.F, s.gp, s.alpha = f32(s.F), f32(s.gp), f32(s.alpha)
        rounds += 1
    # a8: final pass at the accepted dwell weights in plain fp32 (the library's final pass is the SIMT kernel)
    Xf = np.stack([s.x for s in states]).astype(f32)
    dose = (Xf.astype(np.float64) ** 2 @ mc.D.astype(np.float64).T).astype(f32)
    starts = np.cumsum([0] + [((s.n_points + 63) // 64) * 64 for s in c.structures[:-1]])
    dose_u = np.concatenate([dose[:, o:o + s.n_points] for o, s in zip(starts, c.structures)], axis=1)
    F_final, _ = mc.evaluate(Xf, w)
    dvh = np.stack([oracle.dvh(dose_u[k].astype(np.float64), c.structures, c.rx) for k in range(K)])
    return dict(F=F_final.astype(np.float64), iters_done=np.array([s.it for s in states]), dvh=dvh, rounds=rounds,
                status=np.array([s.status for s in states]))


@pytest.mark.parametrize("name,kw,iters", [("C1", {}, 50),
                                            ("C2", dict(counts=(700, 160, 170, 170), n_plans=12), 60)])
def test_modelled_tensor_route_meets_the_parity_bar_after_a_full_optimisation(name, kw, iters):
    c = gc.make_case(name, **kw)
    ref = oracle.optimize(c.D, c.structures, c.rx, c.T0, c.weights, m=c.m, iters=iters)
    out = optimise_model(c, iters)
    assert (out["iters_done"] == ref["iters_done"]).all() and (out["status"] == ref["status"]).all()
    assert (np.abs(out["F"] - ref["F"]) / ref["F"]).max() < 1e-3
    assert np.abs(out["dvh"] - ref["dvh"]).max() < 0.5
    assert out["rounds"] >= 1 + iters
