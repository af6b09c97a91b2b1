"""-m gpu_optional: gmco_options.dose_kernel = 2 -- the gradient contraction on CTA pairs (k_grad_tc_pair).
The option is off by default and has run on the CPU emulation only (tests/test_emu_kernels.py), so its GPU tests carry the
marker gpu_optional: neither -m gpu nor -m "not gpu" selects them (`python -m pytest tests -m gpu_optional`).  Bars:
north_star's 1e-4 per evaluation, and the same bits as k_grad_tc where both sum in the same order."""
import numpy as np
import pytest

import gmco_cases as gc
import oracle

pytestmark = pytest.mark.gpu_optional
TOL = 1e-4


@pytest.fixture(scope="module")
def g():
    import torch
    assert torch.cuda.is_available(), "GPU tests need a B200"
    import paper_1904_01567_b200 as g
    from paper_1904_01567_b200 import build
    build.build()
    return g


def _evaluate(g, c, T, dose_kernel):
    h = g.gmco_create(c.D, c.structures, c.rx, g.binding.make_options(m=c.m, dose_kernel=dose_kernel))
    try:
        return g.gmco_evaluate(h, T, c.weights, want_dose=True, want_grad=True, host=True)
    finally:
        g.gmco_destroy(h)


@pytest.mark.parametrize("n_cath,n_pos,n_plans", [(4, 10, 256), (18, 14, 256), (17, 14, 500)], ids=["A40", "A252", "A238_4_tiles"])
def test_pair_gradient_kernel_matches_the_oracle_and_the_single_cta_kernel(g, n_cath, n_pos, n_plans):
    c = gc.make_case("C1", n_cath=n_cath, n_pos=n_pos, counts=(900, 210, 300, 270), n_plans=n_plans, seed_points=5, seed_weights=6)
    q = g.gmco_tc_schedule(c.n_dwell, [s.n_points for s in c.structures], c.n_plans, 148, 2)
    assert q["grad_pair"] == 1
    T = np.repeat(c.T0[None], c.n_plans, axis=0) * np.linspace(0.6, 1.4, c.n_plans)[:, None].astype(np.float32)
    ref = oracle.evaluate(c.D, c.structures, T, c.weights)
    out, base = _evaluate(g, c, T, 2), _evaluate(g, c, T, 0)
    gn = np.linalg.norm(out["grad_x"] - ref["grad_x"], axis=1) / np.linalg.norm(ref["grad_x"], axis=1)
    assert gn.max() < TOL and (np.abs(out["F"] - ref["F"]) / ref["F"]).max() < TOL
    assert (out["grad_x"] == base["grad_x"]).all() and (out["dose"] == base["dose"]).all()      # same products, same order


def test_c3_full_size_and_optimisation_with_compaction(g):
    c = gc.make_case("C3")
    T = np.repeat(gc.random_starts(c, 1, seed=100), c.n_plans, axis=0) * np.linspace(0.5, 1.5, c.n_plans)[:, None].astype(np.float32)
    out, base = _evaluate(g, c, T, 2), _evaluate(g, c, T, 0)
    assert (out["grad_x"] == base["grad_x"]).all()
    c1 = gc.make_case("C1", n_plans=512)
    ref = oracle.optimize(c1.D, c1.structures, c1.rx, c1.T0, c1.weights, m=c1.m, iters=200, eps=1e-4)
    h = g.gmco_create(c1.D, c1.structures, c1.rx, g.binding.make_options(m=c1.m, eps=1e-4, dose_kernel=2))
    try:
        g.gmco_optimize(h, c1.T0, c1.weights, 200)
        a = g.gmco_result(h, host=True)
    finally:
        g.gmco_destroy(h)
    d_it = a["iters_done"] - ref["iters_done"]
    assert (a["plan_status"] == 1).all() and (d_it == 0).mean() > 0.7
    hit = d_it == 0
    assert (np.abs(a["objective"][hit] - ref["F"][hit]) / ref["F"][hit]).max() < 1e-3
