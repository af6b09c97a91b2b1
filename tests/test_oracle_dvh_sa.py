"""Pins of the oracle's DVH indices (A17) and SA chain (config 5, c.5)."""
from pathlib import Path

import numpy as np
import pytest

import gmco_cases as gc
import oracle


def test_d10_nearest_rank_on_ten_known_doses():
    st = [gc.Structure("u", 10, -np.inf, 16.5, 1, 1, gc.DVH_D, 10.0)]
    dose = np.array([3, 9, 1, 10, 4, 2, 8, 7, 5, 6], float)
    assert oracle.dvh(dose, st, 10.0)[0] == pytest.approx(100.0)     # hottest of 10 -> 10 Gy = 100 % of Rx 10
    st[0].dvh_level = 30.0
    assert oracle.dvh(dose, st, 10.0)[0] == pytest.approx(80.0)      # 3rd hottest = 8


def test_rank_is_ceil_of_fraction():
    st = [gc.Structure("u", 7, -np.inf, 1, 1, 1, gc.DVH_D, 10.0)]
    dose = np.arange(1.0, 8.0)
    assert oracle.dvh(dose, st, 1.0)[0] == pytest.approx(700.0)      # ceil(0.7) = 1 -> hottest
    st = [gc.Structure("u", 21, -np.inf, 1, 1, 1, gc.DVH_D, 10.0)]
    dose = np.arange(1.0, 22.0)
    assert oracle.dvh(dose, st, 1.0)[0] == pytest.approx(1900.0)     # ceil(2.1) = 3 -> 19


def test_v100_counts_ties_as_covered_and_skips_other_structures():
    st = [gc.Structure("p", 4, 15, 22.5, 1, 1, gc.DVH_V, 100.0),
          gc.Structure("x", 2, -np.inf, 1, 1, 1, gc.DVH_NONE, 0.0),
          gc.Structure("r", 4, -np.inf, 11.25, 1, 1, gc.DVH_V, 75.0)]
    dose = np.array([15.0, 14.999999, 20.0, 3.0, 99.0, 99.0, 11.25, 11.2, 12.0, 0.0])
    out = oracle.dvh(dose, st, 15.0)
    assert out == pytest.approx([50.0, 0.0, 50.0])


def _sa_hand_case():
    import gmco_cases as gc
    D = np.array([[1.0, 0.0], [0.0, 2.0]], np.float32)
    st = [gc.Structure("A", 1, 10.0, np.inf, 1.0, 0.0, 0, 0.0), gc.Structure("B", 1, -np.inf, 4.0, 0.0, 1.0, 0, 0.0)]
    w = np.array([[1.0, 0.0], [0.0, 1.0]], np.float32)
    rows = [ln.split() for ln in (Path(__file__).parent / "golden" / "sa_chain_hand_case.txt").read_text().splitlines()
            if ln and not ln.startswith("#")]
    assert rows[0] == "scenario n j z u t0 t1 F n_accepted".split()
    rows = [[float(v) for v in r] for r in rows[1:]]
    setup = {1: dict(T0=np.array([8.0, 1.0], np.float32), temp0=2.0, cooling=0.5),
             2: dict(T0=np.array([10.0, 2.0], np.float32), temp0=1.0, cooling=0.995)}
    return D, st, w, rows, setup


@pytest.mark.parametrize("scenario", [1, 2])
def test_sa_move_clip_floor_metropolis_and_cooling_against_the_hand_worked_chain(scenario):
    """tests/golden/sa_chain_hand_case.txt: downhill accept, uphill accept with u just below exp(-dF/T_n), uphill reject
    with u just above, a move clipped at 0, a move whose width is the 0.01 tau floor, and T_n = temp0 cooling^n at
    n = 0..3 bracketed from both sides.  State after every prefix of the chain (BASELINE.json configs[4])."""
    D, st, w, rows, setup = _sa_hand_case()
    rows = [r for r in rows if int(r[0]) == scenario]
    cfg = setup[scenario]
    j = np.array([r[2] for r in rows], np.int32); z = np.array([r[3] for r in rows]); u = np.array([r[4] for r in rows])
    assert [int(r[1]) for r in rows] == list(range(len(rows)))
    for n, r in enumerate(rows):
        out = oracle.sa_chain(D, st, w, cfg["T0"], 5.0, j[:n + 1], z[:n + 1], u[:n + 1], temp0=cfg["temp0"], cooling=cfg["cooling"])
        assert out["t"] == pytest.approx([r[5], r[6]], rel=1e-12, abs=1e-15), f"dwell times after step {n}"
        assert out["F"] == pytest.approx(r[7], rel=1e-12, abs=1e-15), f"objective after step {n}"
        assert out["n_accepted"] == int(r[8]), f"accepted moves after step {n}"


def _draws(case, steps, seed):
    rng = np.random.Generator(np.random.PCG64(seed))
    return (rng.integers(0, case.n_dwell, steps).astype(np.int32), rng.standard_normal(steps),
            rng.random(steps))


def test_sa_incremental_dose_equals_recomputed_dose(case_small):
    c = case_small
    j, z, u = _draws(c, 3000, 1)
    r = oracle.sa_chain(c.D, c.structures, c.weights[0], c.T0, float(c.T0[0]), j, z, u, want_dose=True)
    d = c.D.astype(np.float64) @ r["t"]
    assert r["dose"] == pytest.approx(d, rel=1e-11)
    assert (r["t"] >= 0).all() and 0 < r["n_accepted"] <= 3000
    F = oracle.eval_plan(c.D, c.structures, c.weights[0], np.sqrt(r["t"]))["F"]
    assert r["F"] == pytest.approx(F, rel=1e-10)


def test_sa_at_zero_temperature_never_goes_uphill(case_small):
    c = case_small
    F_prev = oracle.evaluate(c.D, c.structures, c.T0, c.weights[:1])["F"][0]
    for steps in (50, 200, 800):
        j, z, u = _draws(c, steps, 2)
        F = oracle.sa_chain(c.D, c.structures, c.weights[0], c.T0, float(c.T0[0]), j, z, u, temp0=0.0)["F"]
        assert F <= F_prev
        F_prev = F


def test_sa_approaches_the_lbfgs_objective(case_small):
    """SA and L-BFGS reach the same objective (here within a loose band)."""
    c = case_small
    j, z, u = _draws(c, 20000, 3)
    sa = oracle.sa_chain(c.D, c.structures, c.weights[0], c.T0, float(c.T0[0]), j, z, u)
    lb = oracle.optimize(c.D, c.structures, c.rx, c.T0, c.weights[:1], m=10, iters=400)["F"][0]
    assert lb * (1 - 1e-6) <= sa["F"] <= lb * 1.05
