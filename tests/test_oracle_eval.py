"""Pins of the oracle's single evaluation (dose, penalty, objective, gradient).

Each test ties orc_eval_plan to something that is NOT the oracle itself: a
hand-worked fixture, brute force in exact rational arithmetic, a closed form,
an invariant of Eqs. 1-4, or finite differences.
"""
from fractions import Fraction
from pathlib import Path

import numpy as np
import pytest

import gmco_cases as gc
import oracle

GOLDEN = Path(__file__).parent / "golden"


def _golden(name):
    out = {}
    for line in (GOLDEN / name).read_text().splitlines():
        if line.startswith("#") or line.startswith("key") or not line.strip():
            continue
        k, v = line.split()
        out[k] = float(v)
    return out


def test_hand_worked_2x2_case():
    """tests/golden/eq1_eq2_hand_case.txt: Eqs. 1-4 by pencil."""
    g = _golden("eq1_eq2_hand_case.txt")
    D = np.array([[1, 2], [3, 4]], dtype=np.float32)
    st = [gc.Structure("A", 1, 2.0, 3.0, 3.0, 5.0, 0, 0.0), gc.Structure("B", 1, 1.0, 2.0, 3.0, 5.0, 0, 0.0)]
    w = np.array([[0.5, 0.5], [2.0, 2.0]], dtype=np.float32)
    r = oracle.eval_plan(D, st, w, np.sqrt([0.5, 0.25]))
    assert r["dose"] == pytest.approx([g["d0"], g["d1"]], abs=1e-15)
    assert r["F"] == pytest.approx(g["F"], rel=1e-15)
    assert r["Fterm"][0, 0] == pytest.approx(g["fterm_A_lo"]) and r["Fterm"][0, 1] == 0
    assert r["Fterm"][1, 1] == pytest.approx(g["fterm_B_hi"]) and r["Fterm"][1, 0] == 0
    assert r["r"] == pytest.approx([g["r0"], g["r1"]], rel=1e-15)
    assert r["g"] == pytest.approx([g["g0"], g["g1"]], rel=1e-14)


def test_dose_matches_exact_rational_brute_force(case_small):
    """Eq. 1 as a triple loop in exact rationals (a transposed or dropped index fails)."""
    c = case_small
    rng = np.random.default_rng(3)
    T = rng.uniform(0, 3, size=(2, c.n_dwell)).astype(np.float32)
    out = oracle.evaluate(c.D, c.structures, T, c.weights[:2])
    for k in range(2):
        for i in (0, 7, 119, 120, 159, 259):
            exact = sum(Fraction(float(c.D[i, l])) * Fraction(float(T[k, l])) for l in range(c.n_dwell))
            # x = sqrt(t) then t = x*x: one rounding each way in fp64
            assert out["dose"][i, k] == pytest.approx(float(exact), rel=1e-13)


def test_uniform_start_mean_prostate_dose_is_rx(case_c1):
    """Closed form of reading A7: tau = Rx / mean_i sum_l D_il."""
    c = case_c1
    out = oracle.evaluate(c.D, c.structures, c.T0, c.weights[:1])
    assert out["dose"][:800, 0].mean() == pytest.approx(c.rx, rel=1e-6)


def test_zero_penalty_plan_has_zero_everything(case_small):
    """Thresholds enclosing every dose -> F = 0, r = 0, g = 0 exactly (Eq. 2 middle branch)."""
    c = case_small
    d = c.D.astype(np.float64) @ c.T0.astype(np.float64)
    st, o = [], 0
    for s in c.structures:
        dd = d[o:o + s.n_points]; o += s.n_points
        st.append(gc.Structure(s.name, s.n_points, dd.min() - 1e-6, dd.max() + 1e-6, 2.0, 3.0, 0, 0.0))
    w = np.ones((1, 4, 2), np.float32)
    out = oracle.evaluate(c.D, st, c.T0, w)
    assert out["F"][0] == 0.0 and (out["grad_x"] == 0).all() and (out["G"] == 0).all()
    res = oracle.optimize(c.D, st, c.rx, c.T0, w, m=5, iters=20)
    assert res["iters_done"][0] == 0 and res["status"][0] == 1
    assert res["T"][0] == pytest.approx(c.T0.astype(np.float64), rel=1e-15)


def test_each_branch_of_eq2_and_the_boundaries():
    """d exactly at D_min / D_max gives 0 (Eq. 2 uses strict inequalities)."""
    D = np.eye(4, dtype=np.float32)
    st = [gc.Structure("s", 4, 2.0, 3.0, 7.0, 11.0, 0, 0.0)]
    w = np.array([[1.0, 1.0]], np.float32)
    r = oracle.eval_plan(D, st, w, np.sqrt([1.5, 2.0, 3.0, 4.0]))
    # f = 7*(0.5)^2, 0, 0, 11*(1)^2 ; mean over 4 points
    assert r["F"] == pytest.approx((7 * 0.25 + 11 * 1.0) / 4, rel=1e-14)
    assert r["r"] == pytest.approx([2 * 7 * (-0.5) / 4, 0, 0, 2 * 11 * 1.0 / 4], rel=1e-14)


def test_disabled_sides_with_infinite_thresholds():
    D = np.eye(2, dtype=np.float32)
    st = [gc.Structure("s", 2, -np.inf, 1.0, 5.0, 2.0, 0, 0.0)]
    r = oracle.eval_plan(D, st, np.array([[9.0, 1.0]], np.float32), np.sqrt([0.1, 3.0]))
    assert r["F"] == pytest.approx(2.0 * 4.0 / 2) and np.isfinite(r["g"]).all()


def test_objective_is_linear_in_weights_and_nonnegative(case_small):
    c = case_small
    T = gc.random_starts(c, 3, seed=5)
    a = oracle.evaluate(c.D, c.structures, T, c.weights[:3])
    b = oracle.evaluate(c.D, c.structures, T, 2.5 * c.weights[:3])
    assert (a["F"] >= 0).all() and (a["F"] > 0).any()
    assert b["F"] == pytest.approx(2.5 * a["F"], rel=1e-6)          # fp32 rounding of 2.5*w
    assert b["grad_x"] == pytest.approx(2.5 * a["grad_x"], rel=1e-5, abs=1e-9)
    assert a["Fterm"].sum(axis=(1, 2)) == pytest.approx(a["F"], rel=1e-14)


def test_permuting_points_inside_a_structure_leaves_F_and_g_unchanged(case_small):
    c = case_small
    rng = np.random.default_rng(11)
    perm = np.arange(c.n_points); o = 0
    for s in c.structures:
        perm[o:o + s.n_points] = o + rng.permutation(s.n_points); o += s.n_points
    T = gc.random_starts(c, 2, seed=6)
    a = oracle.evaluate(c.D, c.structures, T, c.weights[:2])
    b = oracle.evaluate(c.D[perm], c.structures, T, c.weights[:2])
    assert b["F"] == pytest.approx(a["F"], rel=1e-12)
    assert b["grad_x"] == pytest.approx(a["grad_x"], rel=1e-10, abs=1e-12)
    assert b["dose"] == pytest.approx(a["dose"][perm], rel=0, abs=0)


def test_gradient_matches_central_finite_differences(case_small):
    """Eq. 3 against Eq. 2/4: F is C^1, so central differences are valid everywhere."""
    c = case_small
    rng = np.random.default_rng(2)
    for k in range(3):
        x = np.sqrt(rng.uniform(0.2, 2.0, c.n_dwell) * float(c.T0[0]))
        base = oracle.eval_plan(c.D, c.structures, c.weights[k], x)
        assert base["F"] > 0
        h = 1e-6
        fd = np.empty_like(x)
        for l in range(c.n_dwell):
            xp, xm = x.copy(), x.copy(); xp[l] += h; xm[l] -= h
            fd[l] = (oracle.eval_plan(c.D, c.structures, c.weights[k], xp)["F"]
                     - oracle.eval_plan(c.D, c.structures, c.weights[k], xm)["F"]) / (2 * h)
        err = np.linalg.norm(fd - base["g"]) / np.linalg.norm(base["g"])
        assert err < 1e-7, err


def test_chain_rule_identity(case_small):
    """Eq. 3 summed over points: g = 2 x o (D^T r), with numpy doing the contraction."""
    c = case_small
    x = np.sqrt(gc.random_starts(c, 1, seed=9)[0].astype(np.float64))
    r = oracle.eval_plan(c.D, c.structures, c.weights[1], x)
    G = c.D.astype(np.float64).T @ r["r"]
    assert r["G"] == pytest.approx(G, rel=1e-12, abs=1e-15)
    assert r["g"] == pytest.approx(2 * x * G, rel=1e-12, abs=1e-15)
    assert r["dose"] == pytest.approx(c.D.astype(np.float64) @ (x * x), rel=1e-13)


def test_plan_independence(case_small):
    c = case_small
    T = gc.random_starts(c, 4, seed=1)
    batch = oracle.evaluate(c.D, c.structures, T, c.weights)
    for k in range(4):
        one = oracle.evaluate(c.D, c.structures, T[k:k + 1], c.weights[k:k + 1])
        assert one["F"][0] == batch["F"][k] and (one["grad_x"][0] == batch["grad_x"][k]).all()


def test_line_search_polynomial_identity(case_small):
    """d(x + a p) = d + 2a D(x o p) + a^2 D(p o p): the linearity the CUDA path may exploit."""
    c = case_small
    rng = np.random.default_rng(4)
    x = np.sqrt(rng.uniform(0.5, 1.5, c.n_dwell)); p = rng.normal(size=c.n_dwell) * 0.2
    Dd = c.D.astype(np.float64)
    for a in (1.0, 0.5, 0.125):
        lhs = oracle.eval_plan(c.D, c.structures, c.weights[0], x + a * p)["dose"]
        rhs = Dd @ (x * x) + 2 * a * (Dd @ (x * p)) + a * a * (Dd @ (p * p))
        assert lhs == pytest.approx(rhs, rel=1e-12)


def test_line_search_polynomial_slope_identity(case_small):
    """phi'(alpha) = grad F(x + alpha p) . p = sum_i dF/dd_i (2 a_i + 2 alpha b_i) with a = D(x o p), b = D(p o p): what the
    optional polynomial line search (kernels_ls.cu) uses for the slope condition of the approximate test, written with
    the oracle's r = dF/dd and gradient."""
    c = case_small
    rng = np.random.default_rng(5)
    x = np.sqrt(rng.uniform(0.5, 1.5, c.n_dwell)); p = rng.normal(size=c.n_dwell) * 0.2
    Dd = c.D.astype(np.float64)
    a_col, b_col = Dd @ (x * p), Dd @ (p * p)
    for al in (1.0, 0.5, 0.25, 0.0625):
        ev = oracle.eval_plan(c.D, c.structures, c.weights[0], x + al * p)
        assert ev["g"] @ p == pytest.approx(ev["r"] @ (2 * a_col + 2 * al * b_col), rel=1e-10)


def test_structure_sizes_must_add_up(case_small):
    c = case_small
    with pytest.raises(ValueError):
        oracle.evaluate(c.D[:-1], c.structures, c.T0, c.weights[:1])
