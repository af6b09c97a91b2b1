"""Input generator: shapes, determinism, the A7 closed form, K-sharding."""
import numpy as np

import gmco_cases as gc


def test_shapes_and_determinism():
    a = gc.make_case("C1"); b = gc.make_case("C1")
    assert a.D.shape == (1500, 40) and a.D.dtype == np.float32
    assert a.weights.shape == (8, 4, 2) and a.T0.shape == (40,)
    assert [s.n_points for s in a.structures] == [800, 200, 250, 250]
    assert a.sha256() == b.sha256()
    assert gc.make_case("C1", seed_points=5).sha256() != a.sha256()
    assert (a.D > 0).all() and np.isfinite(a.D).all()


def test_geometry_inside_bounds():
    c = gc.make_case("C1")
    p = c.points
    e = (p[:800, 0] / gc.AX) ** 2 + (p[:800, 1] / gc.AY) ** 2 + (p[:800, 2] / gc.AZ) ** 2
    assert (e <= 1).all() and (np.hypot(p[:800, 0], p[:800, 1]) > gc.URETHRA_R).all()
    assert (np.hypot(p[800:1000, 0], p[800:1000, 1]) <= gc.URETHRA_R).all()
    assert (p[1000:1250, 1] <= -17.5).all() and (p[1250:, 2] >= gc.AZ).all()
    dw = c.dwell
    e = (dw[:, 0] / gc.AX) ** 2 + (dw[:, 1] / gc.AY) ** 2 + (dw[:, 2] / gc.AZ) ** 2
    assert (e < 1).all() and (np.hypot(dw[:, 0], dw[:, 1]) >= gc.CATH_MIN_R - 1e-9).all()


def test_radial_function_is_normalised_and_bounded():
    r = np.linspace(0.1, 8, 500)
    g = gc.radial_g(r)
    assert abs(gc.radial_g(np.array([1.0]))[0] - 1.0) < 1e-15
    assert g.min() > 0.7 and g.max() < 1.01


def test_weights_layout_and_range():
    w = gc.hidden_weights(64, 7)
    assert (w[:, 1:, 0] == 0).all()                      # organs at risk have no under-dose term
    nz = np.concatenate([w[:, 0, :].ravel(), w[:, 1:, 1].ravel()])
    assert nz.min() >= 0.1 * (1 - 1e-6) and nz.max() <= 10 * (1 + 1e-6)


def test_uniform_start_gives_rx_mean_prostate_dose():
    c = gc.make_case("C2")
    d = c.D[:3500].astype(np.float64) @ c.T0.astype(np.float64)
    assert abs(d.mean() / c.rx - 1) < 1e-6               # fp32 rounding of tau only


def test_shard_plans_partitions_exactly():
    for K, W in [(1000, 8), (7, 3), (5, 8), (0, 2)]:
        spans = [gc.shard_plans(K, W, r) for r in range(W)]
        assert spans[0][0] == 0 and spans[-1][1] == K
        assert all(spans[i][1] == spans[i + 1][0] for i in range(W - 1))
        sizes = [e - b for b, e in spans]
        assert max(sizes) - min(sizes) <= 1
