"""Host-side model of k_step's ROUND protocol (csrc/kernels_lbfgs.cu, rows a6 / a7 of SURVEY 8) held to the oracle.

The kernels do not run an L-BFGS loop per plan: the batch advances in rounds, and in every round a plan has exactly
one trial point evaluated (by the contraction kernels) before k_step decides -- start point (trials = -1), accept
(history push into a ring with head `hh` and count `hc`, two-loop recursion over ring slots, gamma of the newest pair,
restart on a non-descent direction, eps rule, iteration budget) or reject (halve alpha along the same p, stall after
max_trials).  This file restates that state machine in numpy fp64, slot arithmetic and all, drives it with the oracle's
own evaluation and requires the iterates to equal the oracle's loop-per-plan driver: the decomposition into rounds, the
ring indexing and the order of the tests change nothing.  It proves the scheme; the GPU tests prove the code."""
import numpy as np
import pytest

import oracle

RUNNING, ITERS, CONVERGED, STALLED = -1, 0, 1, 2


class PlanState:
    """What k_step keeps per plan between rounds (PlanDev of gmco_internal.cuh)."""

    def __init__(self, x0, m):
        n = x0.size
        self.x, self.xt, self.g, self.p = x0.copy(), x0.copy(), np.zeros(n), np.zeros(n)
        self.S, self.Y = np.zeros((m, n)), np.zeros((m, n))
        self.rho, self.gam = np.zeros(m), np.zeros(m)
        self.F = self.gp = 0.0
        self.alpha, self.it, self.trials, self.hc, self.hh, self.status = 1.0, 0, -1, 0, 0, RUNNING


def k_step_model(s, Ft, gt, m, iters, max_trials, c1, eps, eps_f):
    """One call of k_step for one running plan: (Ft, gt) = objective and gradient at the trial point s.xt."""
    new_dir = False
    if s.trials < 0:                                            # start point: nothing to compare against
        s.x, s.g, s.F = s.xt.copy(), gt.copy(), Ft
        new_dir = True
        if s.it >= iters:
            s.status = ITERS
    else:
        accept = Ft <= s.F + c1 * s.alpha * s.gp
        if not accept and eps_f > 0 and Ft <= s.F + eps_f * abs(s.F):
            accept = gt @ (s.xt - s.x) <= (2 * c1 - 1) * s.alpha * s.gp
        if accept:
            sv, yv = s.xt - s.x, gt - s.g
            sy, ss, yy = sv @ yv, sv @ sv, yv @ yv
            if sy > 1e-10 * np.sqrt(ss) * np.sqrt(yy):          # curvature guard: push into ring slot hh
                s.S[s.hh], s.Y[s.hh] = sv, yv
                s.rho[s.hh], s.gam[s.hh] = 1.0 / sy, sy / yy
                s.hh = 0 if s.hh + 1 == m else s.hh + 1
                s.hc = min(s.hc + 1, m)
            F_old = s.F
            s.x, s.g, s.F = s.xt.copy(), gt.copy(), Ft
            s.it += 1
            new_dir = True
            if eps > 0 and abs(F_old - s.F) <= eps * max(F_old, 1e-30):
                s.status = CONVERGED
            elif s.it >= iters:
                s.status = ITERS
        else:
            s.trials += 1
            if s.trials >= max_trials:
                s.status = STALLED
            else:
                s.alpha *= 0.5
                s.xt = s.x + s.alpha * s.p
    if new_dir:
        gnorm = np.sqrt(s.g @ s.g)
        if s.status == RUNNING and gnorm == 0.0:
            s.status = CONVERGED
        if s.status == RUNNING:
            q = s.g.copy()
            a = np.zeros(m)
            for i in range(s.hc):                               # newest .. oldest
                slot = (s.hh - 1 - i) % m
                a[i] = s.rho[slot] * (s.S[slot] @ q)
                q -= a[i] * s.Y[slot]
            q *= s.gam[(s.hh - 1) % m] if s.hc > 0 else 1.0 / gnorm
            for i in range(s.hc - 1, -1, -1):                   # oldest .. newest
                slot = (s.hh - 1 - i) % m
                b = s.rho[slot] * (s.Y[slot] @ q)
                q += s.S[slot] * (a[i] - b)
            gp = s.g @ -q
            if not gp < 0:                                      # not a descent direction: restart from -g/|g|
                s.hc = 0
                q = s.g / gnorm
                gp = s.g @ -q
            s.p, s.gp, s.alpha, s.trials = -q, gp, 1.0, 0
            s.xt = s.x + s.p


def run_rounds(fg, x0, m, iters, max_trials=20, c1=1e-4, eps=0.0, eps_f=oracle.EPS_F):
    s = PlanState(np.asarray(x0, dtype=np.float64), m)
    rounds = 0
    while s.status == RUNNING and rounds < 1 + iters * (max_trials + 1):
        Ft, gt = fg(s.xt)                                        # the round's contraction kernels
        k_step_model(s, Ft, np.asarray(gt, dtype=np.float64), m, iters, max_trials, c1, eps, eps_f)
        rounds += 1
    return s, rounds


def _fg(c, w):
    def fg(x):
        ev = oracle.eval_plan(c.D, c.structures, w, x)
        return ev["F"], ev["g"]
    return fg


@pytest.mark.parametrize("m,iters,eps", [(5, 40, 0.0), (3, 25, 0.0), (10, 200, 1e-4), (1, 15, 0.0)])
def test_round_protocol_reproduces_the_oracle_driver(case_small, m, iters, eps):
    c = case_small
    for k in range(c.n_plans):
        fg = _fg(c, c.weights[k])
        x0 = np.sqrt(c.T0.astype(np.float64))
        ref = oracle.lbfgs(fg, x0, m=m, iters=iters, eps=eps)
        s, rounds = run_rounds(fg, x0, m, iters, eps=eps)
        assert s.it == ref["iters_done"] and s.status == ref["status"]
        assert s.F == pytest.approx(ref["F"], rel=1e-9)
        assert s.x == pytest.approx(ref["x"], rel=1e-6, abs=1e-8)       # summation order of the dot products differs (numpy vs C loops)
        assert rounds == ref["n_evals"]                         # one evaluation per round: start point + every trial


def test_round_protocol_on_the_driver_pins():
    """The same closed-form pins that pin the oracle's driver, through the round protocol."""
    rng = np.random.default_rng(0)
    Q, _ = np.linalg.qr(rng.normal(size=(10, 10)))
    A = Q @ np.diag(np.geomspace(1.0, 50.0, 10)) @ Q.T
    A = (A + A.T) / 2
    b = rng.normal(size=10)
    fg = lambda x: (0.5 * x @ A @ x - b @ x, A @ x - b)
    s, _ = run_rounds(fg, np.zeros(10), 10, 150)
    assert s.x == pytest.approx(np.linalg.solve(A, b), rel=1e-6, abs=1e-7)
    # x^4 from 0.5: the unit step to -0.5 gives equal F (rejected), alpha = 1/2 lands on 0
    s, rounds = run_rounds(lambda x: (float(x[0] ** 4), np.array([4 * x[0] ** 3])), np.array([0.5]), 3, 1)
    assert s.x[0] == pytest.approx(0.0, abs=1e-16) and rounds == 3 and s.it == 1
    # a zero gradient at the start freezes the plan before any division (reading A9)
    s, rounds = run_rounds(lambda x: (0.0, np.zeros(2)), np.ones(2), 4, 10)
    assert s.status == CONVERGED and s.it == 0 and rounds == 1
    # a direction that never decreases F stalls after max_trials halvings, x unchanged
    s, rounds = run_rounds(lambda x: (float(abs(x[0] - 1.0)) + (x[0] != 1.0) * 1.0, np.array([1.0])), np.array([1.0]), 2, 5, max_trials=4)
    assert s.status == STALLED and s.x[0] == 1.0 and rounds == 1 + 4
