"""-m gpu: Pareto filter and plan selection (NEXT rows 3-4 of SURVEY.md 8(f)) against the oracle: integer results,
compared bit-exactly on the same fp32 inputs -- random pools with many ties, the C1 pool's own results, and the
edge cases (empty pool, one plan, all plans equal, NaN objective)."""
import numpy as np
import pytest

import gmco_cases as gc
import oracle

pytestmark = pytest.mark.gpu

CRIT = [(0, +1, 90.0, 95.0, 0), (1, -1, 118.0, 118.0, 1), (2, -1, 10.0, 10.0, 2), (3, -1, 10.0, 10.0, 2)]


@pytest.fixture(scope="module")
def gh(case_c1):
    import torch
    assert torch.cuda.is_available(), "GPU tests need a B200"
    import paper_1904_01567_b200 as g
    from paper_1904_01567_b200 import build
    build.build()
    h = g.gmco_create(case_c1.D, case_c1.structures, case_c1.rx)
    yield g, h
    g.gmco_destroy(h)


@pytest.mark.parametrize("K,M,levels", [(1, 1, 3), (7, 2, 4), (300, 5, 6), (1000, 8, 3), (2500, 5, 50), (513, 16, 2)])
def test_pareto_front_matches_the_definition(gh, K, M, levels):
    g, h = gh
    rng = np.random.Generator(np.random.PCG64(K * 31 + M))
    obj = (rng.integers(0, levels, size=(K, M)) + (rng.random((K, M)) < 0.3) * rng.random((K, M))).astype(np.float32)
    out = g.gmco_pareto_front(h, obj)
    ref = oracle.pareto_front(obj)
    assert (out["nondominated"] == ref).all() and out["n_nondominated"] == int(ref.sum())


def test_pareto_front_edge_cases(gh):
    g, h = gh
    assert g.gmco_pareto_front(h, np.zeros((0, 3), np.float32))["n_nondominated"] == 0
    same = np.full((40, 4), 2.5, np.float32)
    assert g.gmco_pareto_front(h, same)["nondominated"].all()                # equal plans do not dominate each other
    obj = np.array([[1, 1], [np.nan, 0], [2, 2]], np.float32)                # NaN compares false both ways
    assert g.gmco_pareto_front(h, obj)["nondominated"].tolist() == oracle.pareto_front(obj).tolist() == [True, True, False]
    import torch
    dev = torch.rand(777, 5, device="cuda")
    assert (g.gmco_pareto_front(h, dev)["nondominated"] == oracle.pareto_front(dev.cpu().numpy())).all()
    with pytest.raises(g.GmcoError):
        g.gmco_pareto_front(h, np.zeros((4, 17), np.float32))


@pytest.mark.parametrize("K,seed", [(1, 1), (9, 2), (1000, 3), (5000, 4)])
def test_select_plan_matches_the_oracle(gh, K, seed):
    g, h = gh
    rng = np.random.Generator(np.random.PCG64(seed))
    v100 = rng.choice([85., 89.99, 90., 94., 95., 97.5, 99.], size=K)
    d10 = rng.choice([100., 117., 117.99, 118., 125.], size=K)
    oar = rng.choice([0., 2.5, 9.99, 10., 20.], size=(K, 2))
    for regime in ("mixed", "no_plus", "all_invalid", "nobody_meets_target"):
        dvh = np.column_stack([v100, d10, oar]).astype(np.float32)
        if regime == "no_plus": dvh[:, 0] = np.minimum(dvh[:, 0], 94.0)
        if regime == "all_invalid": dvh[:, 2] = 20.0 + rng.integers(0, 3, K)
        if regime == "nobody_meets_target": dvh[:, 0] = 80.0
        out = g.gmco_select_plan(h, dvh, CRIT)
        sel, cls, cnt = oracle.select_plan(dvh, CRIT)
        assert out["selected"] == sel and (out["plan_class"] == cls).all() and (out["class_counts"] == cnt).all(), regime


def test_select_and_pareto_on_the_c1_pool(gh, case_c1):
    """The path as gMCO uses it: optimise a pool, classify, select, count the non-dominated plans."""
    g, h = gh
    c = gc.make_case("C1", n_plans=64)
    g.gmco_optimize(h, c.T0, c.weights, 60)
    res = g.gmco_result(h, host=True)
    out = g.gmco_select_plan(h, res["dvh"], CRIT)
    sel, cls, cnt = oracle.select_plan(res["dvh"], CRIT)
    assert out["selected"] == sel and (out["plan_class"] == cls).all() and (out["class_counts"] == cnt).all()
    terms = res["objective_terms"].reshape(64, -1)
    pf = g.gmco_pareto_front(h, terms)
    assert (pf["nondominated"] == oracle.pareto_front(terms)).all() and pf["n_nondominated"] >= 1
    assert g.gmco_select_plan(h, np.zeros((0, 4), np.float32), CRIT)["selected"] == -1
    with pytest.raises(g.GmcoError):
        g.gmco_select_plan(h, res["dvh"], CRIT[1:])                          # no target criterion
