"""Seeded synthetic HDR-prostate cases (input generator only).

This module serves BOTH the fp64 oracle (``oracle/``) and the CUDA path
(``paper_1904_01567_b200/``).  It holds none of the method's arithmetic
(no dose contraction, no penalty, no optimiser): it only draws geometry and
produces the *input arrays* of the optimisation -- the dose-rate matrix ``D``,
the structure table, the hidden weights and the start dwell times -- with the
shapes of the paper's patient cases (§2.1.1: 16-18 catheters,
N_act 102-385, N_pnt 2753-15998, four organs, 15 Gy).  The paper's 562-case
dataset is not available; these synthetic cases stand in for it.

Recipe = SURVEY.md §8(c) readings A3, A7, A10-A16 and §8(d); restated in
DESIGN.md §3.  Everything is numpy ``Generator(PCG64(seed))``; arrays are
computed in fp64 and rounded once to fp32, so both sides see identical bytes
(``Case.sha256()``).
"""
from __future__ import annotations

import hashlib
from dataclasses import dataclass, field

import numpy as np

# ----------------------------------------------------------------------------
# geometry constants (mm), reading A10: (x, y, z) = (left-right, antero-posterior,
# cranio-caudal); posterior = -y, superior = +z; prostate centred at the origin.
AX, AY, AZ = 22.5, 17.5, 15.0
URETHRA_R = 3.0            # cylinder on the z axis (A13)
CATH_MIN_R = 6.0           # catheters kept >= 6 mm from the urethra axis (A12)
GOLDEN_ANGLE = 2.399963    # Vogel spiral (A12)
RECTUM_Y = (-22.5, -17.5)  # 5 mm slab touching the posterior pole (A13)
RECTUM_HALF_X = 20.0
BLADDER_R = 30.0           # ball resting on the superior pole, lowest 10 mm used (A13)
BLADDER_CAP = 10.0

RX = 15.0                  # Gy
SK_LAMBDA = 0.125          # synthetic S*Lambda in Gy cm^2 / s (A15)
R_FLOOR_CM = 0.1           # r floored at 1 mm (BASELINE.json configs[0])

# Synthetic radial dose function (A14): a smooth 5th-order polynomial in r [cm],
# normalised to g(1 cm) = 1, staying in ~[0.75, 1.0] on 0.1-8 cm.  NOT a
# published source table -- labelled synthetic on purpose.
_G_RAW = np.array([1.0, 0.004, -0.0022, -0.0012, 0.00018, -0.000008], dtype=np.float64)
G_COEF = _G_RAW / _G_RAW.sum()

STRUCT_NAMES = ("prostate", "urethra", "rectum", "bladder")

# dvh_kind codes of include/gmco.h
DVH_NONE, DVH_V, DVH_D = 0, 1, 2


@dataclass
class Structure:
    name: str
    n_points: int
    d_lo: float      # Gy; -inf disables the under-dose side
    d_hi: float      # Gy; +inf disables the over-dose side
    w_lo: float      # base ("class solution") weights
    w_hi: float
    dvh_kind: int    # 0 none | 1 V(level % of Rx) in % of points | 2 D(level % of points) in % of Rx
    dvh_level: float # percent


@dataclass
class Case:
    name: str
    D: np.ndarray                 # [N, A] float32, rows grouped by structure, point-major (Eq. 1)
    structures: list
    rx: float
    weights: np.ndarray           # [K, S, 2] float32 hidden weights (lo, hi) per structure (A3)
    T0: np.ndarray                # [A] float32 uniform start dwell times (A7)
    m: int
    iters: int
    points: np.ndarray = field(repr=False, default=None)   # [N, 3] mm
    dwell: np.ndarray = field(repr=False, default=None)    # [A, 3] mm

    @property
    def n_points(self): return int(self.D.shape[0])
    @property
    def n_dwell(self): return int(self.D.shape[1])
    @property
    def n_plans(self): return int(self.weights.shape[0])
    @property
    def n_structs(self): return len(self.structures)

    def sha256(self) -> str:
        h = hashlib.sha256()
        for a in (self.D, self.weights, self.T0):
            h.update(np.ascontiguousarray(a).tobytes())
        return h.hexdigest()

    def struct_table(self) -> np.ndarray:
        """[S, 7] float64 rows (n_points, d_lo, d_hi, w_lo, w_hi, dvh_kind, dvh_level)."""
        return np.array([[s.n_points, s.d_lo, s.d_hi, s.w_lo, s.w_hi, s.dvh_kind, s.dvh_level]
                         for s in self.structures], dtype=np.float64)


# ----------------------------------------------------------------------------
def catheter_xy(n_cath: int) -> np.ndarray:
    """Seed-free Vogel spiral inside the ellipse, pushed out of the urethra (A12)."""
    c = np.arange(n_cath, dtype=np.float64)
    rho = 0.8 * np.sqrt((c + 0.5) / n_cath)
    th = c * GOLDEN_ANGLE
    xy = np.stack([rho * AX * np.cos(th), rho * AY * np.sin(th)], axis=1)
    rad = np.hypot(xy[:, 0], xy[:, 1])
    scale = np.where(rad < CATH_MIN_R, CATH_MIN_R / np.maximum(rad, 1e-12), 1.0)
    return xy * scale[:, None]


def dwell_positions(n_cath: int, n_pos: int) -> np.ndarray:
    """Catheters parallel to z, n_pos dwell positions each, centred on z = 0 (A11)."""
    xy = catheter_xy(n_cath)
    out = np.empty((n_cath, n_pos, 3), dtype=np.float64)
    j = np.arange(n_pos, dtype=np.float64) - (n_pos - 1) / 2.0
    for c in range(n_cath):
        x, y = xy[c]
        h = AZ * np.sqrt(max(1.0 - (x / AX) ** 2 - (y / AY) ** 2, 0.0))   # half-chord
        step = min(5.0, 2.0 * (h - 1.0) / (n_pos - 1)) if n_pos > 1 else 0.0
        out[c, :, 0], out[c, :, 1], out[c, :, 2] = x, y, j * step
    return out.reshape(n_cath * n_pos, 3)


def _rejection(rng, n, lo, hi, accept):
    """Uniform points in the box [lo, hi] that satisfy accept(); fixed batch size 4n."""
    got, have = [], 0
    lo, hi = np.asarray(lo, float), np.asarray(hi, float)
    while have < n:
        p = lo + (hi - lo) * rng.random((4 * n, 3))
        p = p[accept(p)]
        got.append(p)
        have += len(p)
    return np.concatenate(got)[:n]


def sample_points(rng, n_prostate, n_urethra, n_rectum, n_bladder) -> np.ndarray:
    """Dose points per organ, in the fixed order prostate, urethra, rectum, bladder (A13)."""
    def in_prostate(p):
        e = (p[:, 0] / AX) ** 2 + (p[:, 1] / AY) ** 2 + (p[:, 2] / AZ) ** 2
        return (e <= 1.0) & (np.hypot(p[:, 0], p[:, 1]) > URETHRA_R)
    pr = _rejection(rng, n_prostate, (-AX, -AY, -AZ), (AX, AY, AZ), in_prostate)
    ur = _rejection(rng, n_urethra, (-URETHRA_R, -URETHRA_R, -AZ), (URETHRA_R, URETHRA_R, AZ),
                    lambda p: np.hypot(p[:, 0], p[:, 1]) <= URETHRA_R)
    re = _rejection(rng, n_rectum, (-RECTUM_HALF_X, RECTUM_Y[0], -AZ), (RECTUM_HALF_X, RECTUM_Y[1], AZ),
                    lambda p: np.ones(len(p), bool))
    zc = AZ + BLADDER_R                                   # ball centre, resting on the superior pole
    rc = np.sqrt(BLADDER_R ** 2 - (BLADDER_R - BLADDER_CAP) ** 2)
    bl = _rejection(rng, n_bladder, (-rc, -rc, AZ), (rc, rc, AZ + BLADDER_CAP),
                    lambda p: p[:, 0] ** 2 + p[:, 1] ** 2 + (p[:, 2] - zc) ** 2 <= BLADDER_R ** 2)
    return np.concatenate([pr, ur, re, bl])


def radial_g(r_cm: np.ndarray) -> np.ndarray:
    out = np.zeros_like(r_cm)
    for c in G_COEF[::-1]:
        out = out * r_cm + c
    return out


def dose_rate_matrix(points_mm: np.ndarray, dwell_mm: np.ndarray) -> np.ndarray:
    """INPUT recipe: D_il = S*Lambda * g(r) / r^2, r in cm floored at 0.1 cm; fp64 -> fp32."""
    N, A = len(points_mm), len(dwell_mm)
    D = np.empty((N, A), dtype=np.float32)
    for i0 in range(0, N, 4096):
        d = points_mm[i0:i0 + 4096, None, :] - dwell_mm[None, :, :]
        r = np.maximum(np.sqrt((d * d).sum(-1)) / 10.0, R_FLOOR_CM)
        D[i0:i0 + 4096] = (SK_LAMBDA * radial_g(r) / (r * r)).astype(np.float32)
    return D


def hidden_weights(n_plans: int, seed: int) -> np.ndarray:
    """[K, 4, 2]: five terms per plan, w = 10**U(-1, 1), NOT normalised (A3).

    Term order: prostate-lo, prostate-hi, urethra-hi, rectum-hi, bladder-hi."""
    rng = np.random.Generator(np.random.PCG64(seed))
    w5 = 10.0 ** rng.uniform(-1.0, 1.0, size=(n_plans, 5))
    w = np.zeros((n_plans, 4, 2), dtype=np.float64)
    w[:, 0, 0], w[:, 0, 1] = w5[:, 0], w5[:, 1]
    w[:, 1, 1], w[:, 2, 1], w[:, 3, 1] = w5[:, 2], w5[:, 3], w5[:, 4]
    return w.astype(np.float32)


def default_structures(counts) -> list:
    inf = float("inf")
    npr, nur, nre, nbl = counts
    return [
        Structure("prostate", npr, 15.0, 22.5, 1.0, 1.0, DVH_V, 100.0),   # V100
        Structure("urethra", nur, -inf, 16.5, 1.0, 1.0, DVH_D, 10.0),     # D10
        Structure("rectum", nre, -inf, 11.25, 1.0, 1.0, DVH_V, 75.0),     # V75
        Structure("bladder", nbl, -inf, 11.25, 1.0, 1.0, DVH_V, 75.0),    # V75
    ]


def uniform_start(D: np.ndarray, n_prostate: int, rx: float = RX) -> float:
    """tau such that the mean prostate dose of the uniform start equals Rx (A7)."""
    rows = D[:n_prostate].astype(np.float64).sum(axis=1)
    return float(rx / rows.mean())


# name -> (n_cath, n_pos, (prostate, urethra, rectum, bladder), K, m, iters)
CONFIGS = {
    "C1": (4, 10, (800, 200, 250, 250), 8, 5, 50),
    "C2": (16, 10, (3500, 800, 850, 850), 100, 10, 200),
    "C3": (18, 14, (7000, 1600, 1700, 1700), 1000, 10, 200),
    "C4": (24, 16, (24000, 4000, 6000, 6000), 4096, 10, 100),
}


def make_case(name: str = "C1", *, n_plans: int | None = None, seed_points: int = 1234,
              seed_weights: int = 7, n_cath=None, n_pos=None, counts=None, m=None, iters=None) -> Case:
    """Build one of the BASELINE.json configs (or a custom-sized variant of it)."""
    base = CONFIGS[name] if name in CONFIGS else CONFIGS["C1"]
    n_cath = n_cath or base[0]
    n_pos = n_pos or base[1]
    counts = tuple(counts or base[2])
    K = n_plans if n_plans is not None else base[3]
    m = m or base[4]
    iters = iters if iters is not None else base[5]
    rng = np.random.Generator(np.random.PCG64(seed_points))
    pts = sample_points(rng, *counts)
    dw = dwell_positions(n_cath, n_pos)
    D = dose_rate_matrix(pts, dw)
    tau = uniform_start(D, counts[0])
    return Case(name=name, D=D, structures=default_structures(counts), rx=RX,
                weights=hidden_weights(K, seed_weights),
                T0=np.full(D.shape[1], tau, dtype=np.float32), m=m, iters=iters,
                points=pts, dwell=dw)


def random_starts(case: Case, n: int, seed: int) -> np.ndarray:
    """[n, A] start dwell times U(0, 2 tau) for the convexity test (A7)."""
    rng = np.random.Generator(np.random.PCG64(seed))
    tau = float(case.T0[0])
    return rng.uniform(0.0, 2.0 * tau, size=(n, case.n_dwell)).astype(np.float32)


def shard_plans(n_plans: int, world_size: int, rank: int) -> tuple[int, int]:
    """Contiguous K-shard [begin, end) of rank (plans are independent: DESIGN.md §7)."""
    base, rem = divmod(n_plans, world_size)
    begin = rank * base + min(rank, rem)
    return begin, begin + base + (1 if rank < rem else 0)


def sa_draws(n_dwell: int, n_chains: int, steps: int, seed: int):
    """Random draws of the gSA chains (BASELINE.json configs[4]): the dwell index,
    a standard normal and a uniform per (chain, step).  Inputs of BOTH sides; no method arithmetic."""
    rng = np.random.Generator(np.random.PCG64(seed))
    jdx = rng.integers(0, n_dwell, size=(n_chains, steps), dtype=np.int32)
    z = rng.standard_normal(size=(n_chains, steps))
    u = rng.random(size=(n_chains, steps))
    return jdx, z, u
