"""-m gpu: the CTA-pair dose kernel (k_dose_tc_pair) on shapes the other files do not reach: an even
number of plan tiles with few dwell groups (the run-time ring, `<0, 0>`), an odd number of dwell groups (which the library
keeps on the single-CTA kernel), and the eps rule with compaction over tile PAIRS.  Same tolerances as test_gpu_parity.py."""
import numpy as np
import pytest

import gmco_cases as gc
import oracle

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def g():
    import torch
    assert torch.cuda.is_available(), "GPU tests need a B200"
    import paper_1904_01567_b200 as g
    from paper_1904_01567_b200 import build
    build.build()
    return g


def _eval(g, c, T):
    h = g.gmco_create(c.D, c.structures, c.rx, g.binding.make_options(m=c.m))
    try:
        return g.gmco_evaluate(h, T, c.weights, want_dose=True, want_grad=True, host=True)
    finally:
        g.gmco_destroy(h)


@pytest.mark.parametrize("n_cath,n_pos", [(4, 10), (5, 20), (16, 10)], ids=["A40_2groups_pair", "A100_4groups_pair", "A160_5groups_pair_half_empty_entry"])
def test_pair_kernel_evaluation_parity(g, n_cath, n_pos):
    c = gc.make_case("C1", n_cath=n_cath, n_pos=n_pos, counts=(900, 210, 300, 270), n_plans=256, seed_points=5, seed_weights=6)
    T = np.repeat(c.T0[None], c.n_plans, axis=0) * np.linspace(0.6, 1.4, c.n_plans)[:, None].astype(np.float32)
    ref = oracle.evaluate(c.D, c.structures, T, c.weights)
    out = _eval(g, c, T)
    assert (np.abs(out["dose"] - ref["dose"]) / np.abs(ref["dose"])).max() < 1e-4
    assert (np.abs(out["F"] - ref["F"]) / ref["F"]).max() < 1e-4
    gn = np.linalg.norm(out["grad_x"] - ref["grad_x"], axis=1) / np.linalg.norm(ref["grad_x"], axis=1)
    assert gn.max() < 1e-4


def test_pair_kernel_eps_stop_with_compaction(g):
    c = gc.make_case("C1", n_plans=512)
    eps = 1e-4
    ref = oracle.optimize(c.D, c.structures, c.rx, c.T0, c.weights, m=c.m, iters=200, eps=eps)
    runs = []
    for _ in range(2):
        h = g.gmco_create(c.D, c.structures, c.rx, g.binding.make_options(m=c.m, eps=eps))
        try:
            g.gmco_optimize(h, c.T0, c.weights, 200)
            runs.append(g.gmco_result(h, host=True))
        finally:
            g.gmco_destroy(h)
    a, b = runs
    assert (a["T"] == b["T"]).all() and (a["iters_done"] == b["iters_done"]).all()      # slots vary, numbers do not
    d_it = a["iters_done"] - ref["iters_done"]
    assert (a["plan_status"] == 1).all()
    assert (d_it == 0).mean() > 0.7 and abs(np.median(d_it)) == 0
    hit = d_it == 0
    assert (np.abs(a["objective"] - ref["F"])[hit] / ref["F"][hit] < 1e-3).all()
    assert (np.abs(a["objective"] - ref["F"]) / ref["F"] < 1e-2).all()
