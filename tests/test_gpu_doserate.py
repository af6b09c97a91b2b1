"""-m gpu: the dose-rate matrix kernel (NEXT row 2 of SURVEY.md 8(f), step (i) of PAPER.md:97) against orc_dose_rate,
and the dense DVH point set evaluated once at the end through the existing entry points."""
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


@pytest.mark.parametrize("name", ["C1", "C2", "C3"])
def test_dose_rate_matrix_parity(g, name):
    """fp64 arithmetic on both sides, one rounding to fp32: equal to the last bit almost everywhere, within one fp32
    ulp everywhere (the GPU contracts multiply-adds, the oracle does not)."""
    c = gc.make_case(name, n_plans=1)
    ref = oracle.dose_rate_matrix(c.points, c.dwell, gc.G_COEF, gc.SK_LAMBDA, gc.R_FLOOR_CM)
    D = g.gmco_dose_rate_matrix(c.points, c.dwell, gc.G_COEF, gc.SK_LAMBDA, gc.R_FLOOR_CM, host=True)
    assert D.shape == ref.shape
    assert np.abs(D - ref).max() <= np.spacing(np.abs(ref)).max()
    assert (np.abs(D - ref) <= np.spacing(np.abs(ref))).all()
    assert (D == ref).mean() > 0.999


def test_dose_rate_matrix_edge_cases(g):
    import torch
    rng = np.random.Generator(np.random.PCG64(2))
    p = rng.uniform(-30, 30, (37, 3)).astype(np.float32); q = rng.uniform(-20, 20, (5, 3)).astype(np.float32)
    p[0] = q[0]                                                       # coincident: the floor applies
    ref = oracle.dose_rate_matrix(p, q, [1.0, -0.01], 0.5, 0.1)
    dev = g.gmco_dose_rate_matrix(torch.from_numpy(p).cuda(), torch.from_numpy(q).cuda(), [1.0, -0.01], 0.5, 0.1)
    assert np.abs(dev.cpu().numpy() - ref).max() <= np.spacing(np.abs(ref)).max()
    assert dev[0, 0].item() == pytest.approx(0.5 * (1.0 - 0.001) / 0.01, rel=1e-6)
    assert g.gmco_dose_rate_matrix(p[:0], q, [1.0], 1.0, 0.1, host=True).shape == (0, 5)
    with pytest.raises(g.GmcoError):
        g.gmco_dose_rate_matrix(p, q, [1.0], 1.0, 0.0, host=True)    # r_floor must be positive
    with pytest.raises(g.GmcoError):
        g.gmco_dose_rate_matrix(p, q, [1.0] * 9, 1.0, 0.1, host=True)


def test_optimise_on_the_gpu_made_matrix_and_dense_dvh_set(g):
    """The paper's GPU portions in sequence: dose-rate matrix, optimisation, DVH on a separate, denser
    point set -- the last one as an iters = 0 evaluation of the optimised dwell times on a second handle."""
    c = gc.make_case("C1")
    D = g.gmco_dose_rate_matrix(c.points, c.dwell, gc.G_COEF, gc.SK_LAMBDA, gc.R_FLOOR_CM)
    h = g.gmco_create(D, c.structures, c.rx, g.binding.make_options(m=c.m))
    g.gmco_optimize(h, c.T0, c.weights, c.iters)
    res = g.gmco_result(h, host=True)
    g.gmco_destroy(h)
    ref = oracle.optimize(c.D, c.structures, c.rx, c.T0, c.weights, m=c.m, iters=c.iters)
    assert res["objective"] == pytest.approx(ref["F"], rel=1e-3)
    dense = gc.make_case("C1", counts=(4000, 1000, 1200, 1200), seed_points=4321, n_plans=c.n_plans)
    Dd = g.gmco_dose_rate_matrix(dense.points, c.dwell, gc.G_COEF, gc.SK_LAMBDA, gc.R_FLOOR_CM)
    h2 = g.gmco_create(Dd, dense.structures, c.rx)
    g.gmco_optimize(h2, res["T"], c.weights, 0)
    dvh = g.gmco_result(h2, host=True)["dvh"]
    g.gmco_destroy(h2)
    Dd_ref = oracle.dose_rate_matrix(dense.points, c.dwell, gc.G_COEF, gc.SK_LAMBDA, gc.R_FLOOR_CM)
    dose = Dd_ref.astype(np.float64) @ res["T"].astype(np.float64).T
    ref_dvh = np.stack([oracle.dvh(dose[:, k], dense.structures, c.rx) for k in range(c.n_plans)])
    assert np.abs(dvh - ref_dvh).max() < 0.5
