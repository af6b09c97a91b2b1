"""-m gpu_optional -- deliberately NOT part of `-m gpu`: gmco_options.wide_accum (k_dose_tc<streamed, split main>) has never
run on hardware.  It is the fix chosen on a CPU model for the gradient shortfall of threshold-sitting plans above 256
dwell positions; with it the north_star's 1e-4 is a hard bar here.  It is kept out of the default GPU suite so that an option which is off cannot colour the
record of the default path; run it with `python -m pytest tests -m gpu_optional` on a B200."""
import numpy as np
import pytest

import gmco_cases as gc
import oracle

pytestmark = pytest.mark.gpu_optional        # NOT `gpu`: run with -m gpu_optional (see the module docstring)
TOL = 1e-4


@pytest.fixture(scope="module")
def g():
    import torch
    assert torch.cuda.is_available(), "GPU tests need a B200"
    import paper_1904_01567_b200 as g
    from paper_1904_01567_b200 import build
    build.build()
    return g


@pytest.mark.parametrize("n_cath,n_pos", [(18, 16), (22, 16), (24, 16)])
def test_split_main_meets_1e4_on_threshold_sitting_plans(g, n_cath, n_pos):
    c = gc.make_case("C1", n_cath=n_cath, n_pos=n_pos, counts=(700, 130, 250, 190), n_plans=130, seed_points=9)
    q = g.gmco_tc_schedule(c.n_dwell, [s.n_points for s in c.structures], c.n_plans, 148, 0, 1)
    assert (q["dose_kernel"], q["dose_n_main"], q["dose_tmem_groups"]) == (1, 2, 4)
    worst = np.repeat(c.T0[None], 130, axis=0) * np.linspace(0.6, 1.4, 130)[:, None].astype(np.float32)
    ref = oracle.evaluate(c.D, c.structures, worst, c.weights)
    out = {}
    for wa in (0, 1):
        h = g.gmco_create(c.D, c.structures, c.rx, g.binding.make_options(m=c.m, wide_accum=wa))
        try:
            out[wa] = g.gmco_evaluate(h, worst, c.weights, want_dose=True, want_grad=True, host=True)
        finally:
            g.gmco_destroy(h)
    err = {}
    for wa in (0, 1):
        e_d = (np.abs(out[wa]["dose"] - ref["dose"]) / np.abs(ref["dose"])).max()
        e_f = (np.abs(out[wa]["F"] - ref["F"]) / ref["F"]).max()
        e_g = (np.linalg.norm(out[wa]["grad_x"] - ref["grad_x"], axis=1) / np.linalg.norm(ref["grad_x"], axis=1)).max()
        err[wa] = (e_d, e_f, e_g)
    print(f"A = {c.n_dwell}: (dose, F, grad) one main accumulator {err[0]}, split main {err[1]}")
    assert err[1][0] < TOL and err[1][1] < TOL and err[1][2] < TOL
    assert err[1][0] < err[0][0]                      # the split does cut the dose error


def test_split_main_optimisation_matches_the_oracle(g):
    c = gc.make_case("C1", n_cath=24, n_pos=16, counts=(4200, 900, 1000, 900), n_plans=300, seed_points=21, seed_weights=22, iters=40)
    h = g.gmco_create(c.D, c.structures, c.rx, g.binding.make_options(m=c.m, wide_accum=1))
    try:
        g.gmco_optimize(h, c.T0, c.weights, c.iters)
        out = g.gmco_result(h, host=True)
    finally:
        g.gmco_destroy(h)
    idx = [0, 127, 128, 299]
    ref = oracle.optimize(c.D, c.structures, c.rx, c.T0, c.weights[idx], m=c.m, iters=c.iters)
    assert (np.abs(out["objective"][idx] - ref["F"]) / ref["F"]).max() < 1e-3
    assert np.abs(out["dvh"][idx] - ref["dvh"]).max() < 0.5
