"""Pins of the plan-pool oracle functions (Pareto filter, RTOG classification and selection) against hand-built
cases, brute force by a different route, and invariants -- none of them re-types the function under test."""
import itertools

import numpy as np
import pytest

import oracle

# RTOG 0924 as PAPER.md:132-143 lists it, with "1 cc" expressed as 10 % of the organ's points for these tables:
# (structure, sense, limit_rtog, limit_rtog_plus, role)
CRIT = [(0, +1, 90.0, 95.0, 0), (1, -1, 118.0, 118.0, 1), (2, -1, 10.0, 10.0, 2), (3, -1, 10.0, 10.0, 2)]


def test_pareto_hand_case_two_objectives():
    # (1,5) (2,2) (5,1) form the front; (3,3) is dominated by (2,2); (2,2) twice: equal plans do not dominate each other;
    # (2,6) is dominated by (1,5)
    pts = [(1, 5), (2, 2), (5, 1), (3, 3), (2, 2), (2, 6)]
    assert oracle.pareto_front(pts).tolist() == [True, True, True, False, True, False]


def test_pareto_one_objective_is_the_set_of_minima_and_antichains_survive():
    x = np.array([3.0, 1.0, 2.0, 1.0, 7.0])
    assert oracle.pareto_front(x[:, None]).tolist() == [False, True, False, True, False]
    t = np.linspace(0, 1, 17)
    chain = np.stack([t, 1 - t], axis=1)                      # strict trade-off: nobody dominates anybody
    assert oracle.pareto_front(chain).all()


def test_pareto_against_sorting_sweep_in_two_dimensions():
    """Independent route for M = 2: sort by the first objective, sweep the running minimum of the second."""
    rng = np.random.Generator(np.random.PCG64(3))
    pts = rng.integers(0, 12, size=(200, 2)).astype(np.float32)      # many ties
    ref = np.zeros(len(pts), bool)
    for i, (a, b) in enumerate(pts):
        better_first = pts[:, 0] < a
        same_first = pts[:, 0] == a
        ref[i] = not ((better_first & (pts[:, 1] <= b)).any() or (same_first & (pts[:, 1] < b)).any())
    assert (oracle.pareto_front(pts) == ref).all()


def test_pareto_invariants():
    rng = np.random.Generator(np.random.PCG64(4))
    obj = rng.random((60, 4)).astype(np.float32)
    m = oracle.pareto_front(obj)
    perm = rng.permutation(60)
    assert (oracle.pareto_front(obj[perm]) == m[perm]).all()                       # order of plans is irrelevant
    assert (oracle.pareto_front(obj * np.float32([2, 3, 5, 7])) == m).all()        # positive scaling of a column
    worse = obj[m][0] + np.float32(0.5)                                            # adding a dominated plan changes nothing
    m2 = oracle.pareto_front(np.vstack([obj, worse]))
    assert (m2[:-1] == m).all() and not m2[-1]
    assert m.any()                                                                  # a finite set has a minimal element


def test_selection_priority_order_by_hand():
    #        V100  D10   V75b  V75r
    dvh = [[96.0, 110., 5.0, 5.0],     # RTOG+
           [97.5, 117., 9.0, 9.9],     # RTOG+, higher V100  -> selected
           [92.0, 100., 1.0, 1.0],     # RTOG only
           [99.0, 120., 1.0, 1.0],     # urethra violated
           [97.5, 117., 9.0, 9.9]]     # tie with plan 1 -> lower index wins
    sel, cls, cnt = oracle.select_plan(dvh, CRIT)
    assert sel == 1 and cls.tolist() == [2, 2, 1, 0, 2] and cnt.tolist() == [1, 1, 3]
    sel, cls, cnt = oracle.select_plan(dvh[2:4], CRIT)                 # no RTOG+ plan: the RTOG one
    assert sel == 0 and cls.tolist() == [1, 0]


def test_selection_fallback_among_invalid_plans_by_hand():
    """lowest bladder and rectum V75 while not violating target and urethra."""
    dvh = [[91.0, 110., 12.0, 15.0],   # target + urethra fine, OAR sum 27
           [93.0, 117., 11.0, 10.0],   # target + urethra fine, OAR sum 21 -> selected
           [80.0, 100., 0.0, 0.0],     # lowest OAR sum but target violated
           [95.0, 118., 0.0, 0.0]]     # D10 = 118 is not < 118: urethra violated
    sel, cls, cnt = oracle.select_plan(dvh, CRIT)
    assert sel == 1 and cls.tolist() == [0, 0, 0, 0] and cnt.tolist() == [4, 0, 0]
    sel, _, _ = oracle.select_plan(dvh[2:], CRIT)                      # nobody meets target and urethra: lowest OAR sum overall
    assert sel == 0
    assert oracle.select_plan(np.zeros((0, 4)), CRIT)[0] == -1


def test_selection_boundaries_are_as_the_paper_writes_them():
    """V100 >= 90 % is inclusive, D10 < 118 % and V75 < limit are strict."""
    ok = [[90.0, 117.9, 9.9, 9.9]]
    assert oracle.select_plan(ok, CRIT)[1].tolist() == [1]
    for col, val in ((0, 89.99), (1, 118.0), (2, 10.0), (3, 10.0)):
        bad = [list(ok[0])]; bad[0][col] = val
        assert oracle.select_plan(bad, CRIT)[1].tolist() == [0]
    assert oracle.select_plan([[95.0, 100., 0., 0.]], CRIT)[1].tolist() == [2]


def test_selection_against_exhaustive_enumeration():
    """Brute force by another route: build the full preference order with Python's sort and take its head."""
    rng = np.random.Generator(np.random.PCG64(5))
    vals = {0: [85., 90., 94., 95., 99.], 1: [100., 117., 118., 125.], 2: [0., 5., 10., 20.], 3: [0., 5., 10., 20.]}
    rows = list(itertools.product(*[vals[i] for i in range(4)]))
    for trial in range(40):
        pick = rng.choice(len(rows), size=rng.integers(1, 9), replace=False)
        dvh = np.array([rows[i] for i in pick], dtype=np.float32)

        def rank(k):
            v100, d10, vb, vr = dvh[k]
            rtog = v100 >= 90 and d10 < 118 and vb < 10 and vr < 10
            plus = rtog and v100 >= 95
            core = v100 >= 90 and d10 < 118
            if plus: return (0, -v100, k)
            if rtog: return (1, -v100, k)
            if core: return (2, np.float32(vb) + np.float32(vr), k)
            return (3, np.float32(vb) + np.float32(vr), k)
        order = sorted(range(len(dvh)), key=rank)
        # class 3 plans are only eligible when no class 2 plan exists: the sort order already says so
        assert oracle.select_plan(dvh, CRIT)[0] == order[0]
