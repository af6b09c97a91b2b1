"""Pins of orc_dose_rate (step (i); model: BASELINE.json configs[0]) against closed forms, invariants
and the generator's independent numpy recipe."""
import numpy as np
import pytest

import gmco_cases as gc
import oracle


def test_value_at_one_centimetre_and_inverse_square_law():
    coef = [0.4, 0.3, 0.2, 0.1]                                   # g(1) = 1.0
    q = np.zeros((1, 3), np.float32)
    p = np.array([[10, 0, 0], [0, 20, 0], [0, 0, -40]], np.float32)          # r = 1, 2, 4 cm
    D = oracle.dose_rate_matrix(p, q, coef, 0.125, 0.1)
    assert D[0, 0] == np.float32(0.125)                                       # sk_lambda g(1) / 1^2, exactly
    D1 = oracle.dose_rate_matrix(p, q, [1.0], 2.0, 0.1)                       # g = 1: pure inverse square
    assert D1[:, 0].tolist() == [2.0, 0.5, 0.125]


def test_polynomial_is_evaluated_lowest_power_first():
    q = np.zeros((1, 3), np.float32); p = np.array([[30, 0, 0]], np.float32)  # r = 3 cm
    D = oracle.dose_rate_matrix(p, q, [0.0, 0.0, 1.0], 1.0, 0.1)              # g = r^2 -> D = 1
    assert D[0, 0] == 1.0
    D = oracle.dose_rate_matrix(p, q, [5.0, -1.0], 9.0, 0.1)                  # g = 5 - r = 2 -> D = 9 * 2 / 9
    assert D[0, 0] == 2.0


def test_floor_at_small_radius():
    q = np.zeros((1, 3), np.float32)
    p = np.array([[0, 0, 0], [0.5, 0, 0], [1.0, 0, 0], [2.0, 0, 0]], np.float32)     # 0, 0.05, 0.1, 0.2 cm
    D = oracle.dose_rate_matrix(p, q, [1.0], 1.0, 0.1)
    assert D[:, 0] == pytest.approx([100.0, 100.0, 100.0, 25.0], rel=1e-6)


def test_layout_and_rigid_motion_invariance():
    rng = np.random.Generator(np.random.PCG64(8))
    p = rng.uniform(-30, 30, (50, 3)).astype(np.float32); q = rng.uniform(-20, 20, (7, 3)).astype(np.float32)
    coef = gc.G_COEF
    D = oracle.dose_rate_matrix(p, q, coef, gc.SK_LAMBDA, gc.R_FLOOR_CM)
    assert D.shape == (50, 7)
    Dt = oracle.dose_rate_matrix(q, p, coef, gc.SK_LAMBDA, gc.R_FLOOR_CM)     # swapping the roles transposes D
    assert np.array_equal(Dt, D.T)
    perm = [2, 0, 1]                                                          # relabelling the axes changes nothing
    Dp = oracle.dose_rate_matrix(p[:, perm], q[:, perm], coef, gc.SK_LAMBDA, gc.R_FLOOR_CM)
    assert Dp == pytest.approx(D, rel=1e-6)
    one = oracle.dose_rate_matrix(p[3:4], q[5:6], coef, gc.SK_LAMBDA, gc.R_FLOOR_CM)
    assert one[0, 0] == D[3, 5]                                               # element (i, l) depends on p_i and q_l only


def test_against_the_generators_numpy_recipe(case_c1):
    """gmco_cases.dose_rate_matrix is independent code (vectorised numpy, Horner form): same D to fp32 rounding."""
    c = case_c1
    D = oracle.dose_rate_matrix(c.points, c.dwell, gc.G_COEF, gc.SK_LAMBDA, gc.R_FLOOR_CM)
    assert D.shape == c.D.shape
    assert D == pytest.approx(c.D, rel=5e-6)             # c.D comes from fp64 coordinates, the ABI takes fp32 ones
    p32, q32 = c.points.astype(np.float32).astype(np.float64), c.dwell.astype(np.float32).astype(np.float64)
    D32 = gc.dose_rate_matrix(p32, q32)                  # the recipe on the coordinates the oracle actually saw
    assert D == pytest.approx(D32, rel=2e-7)
    assert (D == D32).mean() > 0.99
