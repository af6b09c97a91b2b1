"""Pins of the oracle's L-BFGS driver and of the whole optimisation (readings A5-A9)."""
import numpy as np
import pytest
import scipy.optimize

import gmco_cases as gc
import oracle


def _spd(n, seed, cond=50.0):
    rng = np.random.default_rng(seed)
    Q, _ = np.linalg.qr(rng.normal(size=(n, n)))
    A = Q @ np.diag(np.geomspace(1.0, cond, n)) @ Q.T
    return (A + A.T) / 2, rng.normal(size=n)


def test_convex_quadratic_reaches_closed_form_minimiser():
    """1/2 x'Ax - b'x, SPD: minimiser A^-1 b (numpy.linalg.solve), F monotone."""
    A, b = _spd(10, 0)
    fg = lambda x: (0.5 * x @ A @ x - b @ x, A @ x - b)
    xs = np.linalg.solve(A, b)
    # Armijo only (eps_f = 0): F is monotone; a function-value line search stalls at
    # |x - x*| ~ sqrt(machine eps), so status 2 is expected
    r = oracle.lbfgs(fg, np.zeros(10), m=10, iters=150, eps_f=0.0)
    assert r["x"] == pytest.approx(xs, rel=1e-6, abs=1e-7)
    assert r["F"] == pytest.approx(-0.5 * b @ xs, rel=1e-12)
    assert (np.diff(r["F_hist"]) <= 0).all()
    assert r["n_skipped"] == 0 and r["status"] in (0, 2) and r["n_approx"] == 0
    # default (reading A5b): the approximate test may pass steps that Armijo cannot resolve;
    # F never rises by more than eps_f |F| per step and the minimiser is reached all the same
    r = oracle.lbfgs(fg, np.zeros(10), m=10, iters=150)
    assert r["x"] == pytest.approx(xs, rel=1e-6, abs=1e-7)
    assert r["F"] == pytest.approx(-0.5 * b @ xs, rel=1e-12)
    h = r["F_hist"]
    assert (np.diff(h) <= oracle.EPS_F * np.abs(h[:-1])).all()


def test_approximate_test_equals_armijo_on_a_quadratic_line():
    """For quadratic phi, phi'(a) <= (2 c1 - 1) phi'(0)  <=>  phi(a) <= phi(0) + c1 a phi'(0):
    with a noise-free objective the two tests take the same decisions, so the iterates agree."""
    A, b = _spd(8, 3, cond=30.0)
    fg = lambda x: (0.5 * x @ A @ x - b @ x, A @ x - b)
    r0 = oracle.lbfgs(fg, np.ones(8), m=5, iters=12, eps_f=0.0)
    r1 = oracle.lbfgs(fg, np.ones(8), m=5, iters=12, eps_f=1e-6)
    assert r1["n_approx"] == 0 and (r0["x"] == r1["x"]).all() and r0["n_evals"] == r1["n_evals"]


def test_approximate_test_accepts_a_step_hidden_by_objective_noise():
    """F quantised to 7 significant digits (an fp32-like objective), exact gradient: near the
    minimum Armijo cannot see the decrease and burns step halvings on every iteration; the
    approximate test accepts those steps at once and ends closer to the minimiser."""
    A, b = _spd(6, 5, cond=20.0)
    xs = np.linalg.solve(A, b)
    def fg(x):
        F = 10.0 + 0.5 * (x - xs) @ A @ (x - xs)
        return float(np.float32(F)), A @ (x - xs)
    r0 = oracle.lbfgs(fg, xs + 1.0, m=6, iters=60, eps_f=0.0)
    r1 = oracle.lbfgs(fg, xs + 1.0, m=6, iters=60, eps_f=1e-6)
    assert r1["n_approx"] > 0 and r1["n_backtracks"] < 5 and r0["n_backtracks"] > 100
    assert np.linalg.norm(r1["x"] - xs) < 0.1 * np.linalg.norm(r0["x"] - xs)


def test_first_step_is_normalised_steepest_descent():
    """Empty history: gamma = 1/|g| so p = -g/|g| and alpha = 1 moves exactly unit length."""
    A = np.diag([1.0, 1.0]); b = np.zeros(2)
    fg = lambda x: (0.5 * x @ A @ x, A @ x)
    r = oracle.lbfgs(fg, np.array([3.0, 4.0]), m=5, iters=1)
    assert r["x"] == pytest.approx([3.0 - 0.6, 4.0 - 0.8], rel=1e-15)
    assert r["n_evals"] == 2 and r["n_backtracks"] == 0


def test_backtracking_halves_until_armijo_holds():
    """F = x^4 from x = 0.5: unit step to -0.5 gives equal F (rejected), alpha = 1/2 lands on 0."""
    fg = lambda x: (float(x[0] ** 4), np.array([4 * x[0] ** 3]))
    r = oracle.lbfgs(fg, np.array([0.5]), m=3, iters=1)
    assert r["n_backtracks"] == 1 and r["x"][0] == pytest.approx(0.0, abs=1e-16)
    assert r["n_bt_iters"] == 1 and r["max_bt_iter"] == 1        # the statistics counters: one iteration, one halving


def test_backtracking_statistics_that_decide_the_line_search_route():
    """a rejected trial step costs ONE more column in the next batched contraction (the plan simply
    rides along), whereas the polynomial route phi(alpha) = F(d + 2 alpha a + alpha^2 b) of SURVEY 8(c.2) costs three
    columns (d is never stored by the fused path, so d, a = D(x o p) and b = D(p o p)) plus the fresh evaluation.  It
    could only pay in iterations with four or more halvings; on the stand-in cases no iteration has more than two, and
    a plan needs 1.0-1.2 halvings per iteration that backtracks at all."""
    worst = 0
    for name, idx in (("C1", slice(None)), ("C2", slice(0, 100, 12))):
        c = gc.make_case(name)
        r = oracle.optimize(c.D, c.structures, c.rx, c.T0, c.weights[idx], m=c.m, iters=c.iters)
        bt, bi, mx = r["n_backtracks"], r["n_bt_iters"], r["max_bt_iter"]
        assert (bi <= bt).all() and (mx <= np.maximum(bt, 0)).all() and ((bt > 0) == (bi > 0)).all()
        assert bt.sum() <= 1.25 * bi.sum()              # halvings per backtracking iteration
        worst = max(worst, int(mx.max()))
        # plan-rounds: what runs (1 + iterations + halvings) against the polynomial route's best case
        now, poly = (1 + c.iters + bt).sum(), (1 + c.iters + bi).sum()
        assert (now - poly) / now < 0.01
    assert worst <= 3


def test_one_dimensional_quadratic_converges_in_two_iterations():
    """After one (s, y) pair the secant equation is exact in 1-D: H = 1/a."""
    fg = lambda x: (2.5 * (x[0] - 3.0) ** 2, np.array([5.0 * (x[0] - 3.0)]))
    r = oracle.lbfgs(fg, np.array([0.0]), m=3, iters=2)
    assert r["x"][0] == pytest.approx(3.0, rel=1e-14)


def test_zero_gradient_start_freezes_immediately():
    fg = lambda x: (0.0, np.zeros_like(x))
    r = oracle.lbfgs(fg, np.ones(3), m=3, iters=5)
    assert r["iters_done"] == 0 and r["status"] == 1 and r["n_evals"] == 1


def test_eps_stops_early_and_looser_eps_stops_sooner():
    A, b = _spd(12, 1, cond=200.0)
    fg = lambda x: (0.5 * x @ A @ x - b @ x + 10.0, A @ x - b)
    its = [oracle.lbfgs(fg, np.zeros(12), m=10, iters=200, eps=e)["iters_done"] for e in (1e-2, 1e-4, 1e-8)]
    assert its[0] <= its[1] <= its[2] < 200 and its[0] < its[2]


def test_matches_scipy_on_rosenbrock_minimum():
    """Library cross-check on a non-quadratic problem: same minimum value as scipy's L-BFGS-B."""
    fg = lambda x: (scipy.optimize.rosen(x), scipy.optimize.rosen_der(x))
    r = oracle.lbfgs(fg, np.full(6, -1.0), m=10, iters=400)
    ref = scipy.optimize.minimize(scipy.optimize.rosen, np.full(6, -1.0), jac=scipy.optimize.rosen_der,
                                  method="L-BFGS-B", options=dict(maxiter=2000, ftol=1e-15, gtol=1e-12))
    assert r["F"] < 1e-12 and ref.fun < 1e-10
    assert r["x"] == pytest.approx(np.ones(6), abs=1e-5)


def test_planted_least_squares_solution(case_c1):
    """One structure, D_lo = D_hi = c, equal weights: Eq. 2 is mean((D t - c)^2).  Rows rescaled so
    that D' t_true = c exactly -> minimum F = 0 at t = t_true."""
    c = case_c1
    rng = np.random.default_rng(8)
    Dp = c.D[:800].astype(np.float64)
    t_true = rng.uniform(0.5, 1.5, c.n_dwell) * float(c.T0[0])
    cval = 15.0
    Dp = (Dp * (cval / (Dp @ t_true))[:, None]).astype(np.float32)
    st = [gc.Structure("target", 800, cval, cval, 1.0, 1.0, 0, 0.0)]
    w = np.ones((1, 1, 2), np.float32)
    f50 = oracle.optimize(Dp, st, c.rx, c.T0, w, m=5, iters=50)["F"][0]
    res = oracle.optimize(Dp, st, c.rx, c.T0, w, m=10, iters=1500)
    assert res["F"][0] < 1e-10 < f50                     # fp32 rounding of D' sets the floor
    assert res["F"][0] < 1e-6 * f50
    assert res["T"][0] == pytest.approx(t_true, rel=2e-3)


def test_random_starts_converge_to_the_same_objective(case_c1):
    """Convexity claim: different starts agree within 0.2 %."""
    c = case_c1
    T0 = gc.random_starts(c, 6, seed=21)
    T0[T0 < 1e-3] = 1e-3                                # a dwell at exactly 0 stays at 0 (A8)
    w = np.repeat(c.weights[2:3], 6, axis=0)
    res = oracle.optimize(c.D, c.structures, c.rx, T0, w, m=10, iters=600)
    ref = oracle.optimize(c.D, c.structures, c.rx, c.T0, w[:1], m=10, iters=600)["F"][0]
    assert np.abs(res["F"] / ref - 1).max() < 2e-3


def test_objective_history_is_monotone_and_stats_consistent(case_c1):
    c = case_c1
    res = oracle.optimize(c.D, c.structures, c.rx, c.T0, c.weights, m=c.m, iters=c.iters, want_hist=True)
    assert (np.diff(res["F_hist"], axis=1) <= 0).all()
    assert (res["iters_done"] == c.iters).all() and (res["status"] == 0).all()
    assert (res["n_evals"] == 1 + c.iters + res["n_backtracks"]).all()
    assert res["F_hist"][:, -1] == pytest.approx(res["F"], rel=1e-14)
    assert (res["F"] < 0.6 * res["F_hist"][:, 0]).all()


def test_final_objective_is_close_to_an_independent_minimiser(case_small):
    """Library cross-check of the END result: scipy L-BFGS-B on a numpy restatement of Eq. 4
    (used only as a bound: the oracle after many iterations must not be above scipy's minimum)."""
    c = case_small
    Dd = c.D.astype(np.float64); w = c.weights[0].astype(np.float64)

    def fg(x):
        d = Dd @ (x * x); F = 0.0; r = np.zeros_like(d); o = 0
        for j, s in enumerate(c.structures):
            dd = d[o:o + s.n_points]
            lo = np.minimum(dd - s.d_lo, 0); hi = np.maximum(dd - s.d_hi, 0)
            F += (w[j, 0] * s.w_lo * lo @ lo + w[j, 1] * s.w_hi * hi @ hi) / s.n_points
            r[o:o + s.n_points] = 2 * (w[j, 0] * s.w_lo * lo + w[j, 1] * s.w_hi * hi) / s.n_points
            o += s.n_points
        return F, 2 * x * (Dd.T @ r)

    ref = scipy.optimize.minimize(fg, np.sqrt(c.T0.astype(np.float64)), jac=True, method="L-BFGS-B",
                                  options=dict(maxiter=5000, ftol=1e-14, gtol=1e-10))
    res = oracle.optimize(c.D, c.structures, c.rx, c.T0, c.weights[:1], m=10, iters=1500)
    assert res["F"][0] == pytest.approx(ref.fun, rel=2e-3)


def test_dwell_starting_at_zero_stays_at_zero(case_small):
    """Reading A8: Eq. 3 vanishes at x_l = 0."""
    c = case_small
    T0 = np.repeat(c.T0[None], 1, axis=0).copy(); T0[0, [3, 17]] = 0.0
    res = oracle.optimize(c.D, c.structures, c.rx, T0, c.weights[:1], m=5, iters=30)
    assert (res["T"][0, [3, 17]] == 0).all() and (res["T"][0] >= 0).all()


def test_polynomial_values_choose_the_step_the_halving_search_accepts(case_small):
    """The optional polynomial line search (csrc/kernels_ls.cu) restated in numpy and held to the oracle:
    along real gL-BFGS trajectories, in every iteration whose first trial step is rejected, the first candidate
    alpha_j = 2^-j that meets the Armijo or the approximate test on the POLYNOMIAL values phi(alpha) = F(d + 2 alpha a +
    alpha^2 b), phi'(alpha) = sum_i dF/dd_i (2 a_i + 2 alpha b_i) -- formed in fp32 as the kernel forms them -- is the step
    the oracle's halving search accepts after evaluating every trial point in full."""
    c = case_small
    D32 = c.D.astype(np.float32)
    n_checked = 0
    for k in range(c.n_plans):
        w = c.weights[k]
        calls = []                                                    # every evaluation the driver asks for, in order

        def fg(x):
            ev = oracle.eval_plan(c.D, c.structures, w, x)
            calls.append((x.copy(), ev["F"], ev["g"].copy()))
            return ev["F"], ev["g"]
        res = oracle.lbfgs(fg, np.sqrt(c.T0.astype(np.float64)), m=5, iters=60)
        # split the call sequence into iterations: a call whose point is x_acc + alpha p with alpha = 1 starts one
        i, x_acc, F_acc, g_acc = 1, calls[0][0], calls[0][1], calls[0][2]
        while i < len(calls):
            p = calls[i][0] - x_acc                                   # the alpha = 1 trial defines the direction
            gp = float(g_acc @ p)
            trials = [calls[i]]
            al = 1.0
            def accepted(t, al):
                return t[1] <= F_acc + 1e-4 * al * gp or (t[1] <= F_acc + oracle.EPS_F * abs(F_acc) and t[2] @ p <= (2e-4 - 1.0) * gp)
            while not accepted(trials[-1], al) and i + 1 < len(calls) and np.allclose(calls[i + 1][0], x_acc + 0.5 * al * p, rtol=0, atol=1e-12):
                i += 1; al *= 0.5; trials.append(calls[i])
            if not accepted(trials[-1], al):
                break                                                 # the run ended inside a line search
            if len(trials) > 1:                                       # the first trial was rejected: the polynomial route's case
                xs, ps = x_acc.astype(np.float32), p.astype(np.float32)
                d = D32 @ (xs * xs); a = D32 @ (xs * ps); b = D32 @ (ps * ps)
                sid = np.repeat(np.arange(len(c.structures)), [s.n_points for s in c.structures])
                dlo = np.array([c.structures[s].d_lo for s in sid], np.float32); dhi = np.array([c.structures[s].d_hi for s in sid], np.float32)
                wl = np.array([w[s, 0] * c.structures[s].w_lo / c.structures[s].n_points for s in sid], np.float32)
                wh = np.array([w[s, 1] * c.structures[s].w_hi / c.structures[s].n_points for s in sid], np.float32)

                def phi(alj):
                    dj = (d + np.float32(2 * alj) * a + np.float32(alj * alj) * b).astype(np.float32)
                    lo, hi = np.minimum(dj - dlo, 0), np.maximum(dj - dhi, 0)
                    val = float((wl * lo * lo + wh * hi * hi).sum(dtype=np.float32))
                    slope = float((2 * (wl * lo + wh * hi) * 2 * (a + np.float32(alj) * b)).sum(dtype=np.float32))
                    return val, slope
                F0 = phi(0.0)[0]
                pick, alj = 0, 1.0
                for j in range(1, 20):
                    alj *= 0.5
                    Fj, sj = phi(alj)
                    if Fj <= F0 + 1e-4 * alj * gp or (Fj <= F0 + oracle.EPS_F * abs(F0) and sj <= (2e-4 - 1.0) * gp):
                        pick = j
                        break
                assert pick == len(trials) - 1, (k, pick, len(trials) - 1)
                n_checked += 1
            x_acc, F_acc, g_acc = trials[-1]
            i += 1
        assert res["iters_done"] > 0
    print("iterations with a rejected first trial checked:", n_checked)
    assert n_checked >= 3                                             # the trajectories do contain rejected first trials
