"""Host-side model of k_result's D_level selection (csrc/kernels_simt.cu, row a8): the rank-th hottest dose is found by a
32-step bisection on the order-preserving unsigned image of fp32 ("largest ordinal o with count(v >= o) >= rank").
Restated in numpy and held bit for bit to the definition the oracle writes out (sort, nearest rank ceil(level n / 100),
reading A17), including ties, negative values, zeros of both signs and the rank clamps.  It proves the scheme; the GPU
tests prove the code."""
import numpy as np
import pytest

import gmco_cases as gc
import oracle


def f2ord(v):
    u = v.astype(np.float32).view(np.uint32)
    return np.where(u & 0x80000000, ~u, u | np.uint32(0x80000000)).astype(np.uint32)


def ord2f(o):
    o = np.uint32(o)
    u = (o & np.uint32(0x7fffffff)) if (o & np.uint32(0x80000000)) else ~o
    return np.array([u], dtype=np.uint32).view(np.float32)[0]


def select_rank(v, rank):
    ords = f2ord(v)
    o = 0
    for bit in range(31, -1, -1):
        cand = o | (1 << bit)
        if int((ords >= np.uint32(cand)).sum()) >= rank:
            o = cand
    return ord2f(o)


def host_rank(n, level):
    r = int(np.ceil(float(n) * float(level) / 100.0))
    return min(max(r, 1), n)


@pytest.mark.parametrize("seed", range(6))
def test_bisection_on_the_ordinal_image_is_the_nearest_rank_selection(seed):
    rng = np.random.default_rng(seed)
    n = int(rng.integers(1, 400))
    v = rng.normal(10.0, 6.0, n).astype(np.float32)
    if seed % 2:
        v[rng.integers(0, n, n // 3 + 1)] = v[0]                  # ties
    if seed == 3:
        v[: n // 2] = 0.0; v[n // 2:] = -0.0                       # zeros of both signs
    for level in (10.0, 50.0, 0.3, 100.0, 99.9):
        rank = host_rank(n, level)
        want = np.sort(v)[::-1][rank - 1]
        got = select_rank(v, rank)
        assert got == want or (got == 0.0 and want == 0.0), (n, level, got, want)
        # and the oracle's DVH routine says the same (in % of Rx)
        st = [gc.Structure("u", n, -np.inf, np.inf, 0.0, 0.0, 2, level)]
        assert oracle.dvh(v.astype(np.float64), st, 15.0)[0] == pytest.approx(100.0 * float(want) / 15.0, rel=1e-12, abs=1e-12)


def test_ordinal_image_preserves_order():
    v = np.array([-np.inf, -3.5, -1e-30, -0.0, 0.0, 1e-30, 2.0, 2.0000002, np.inf], np.float32)
    o = f2ord(v).astype(np.int64)
    assert (np.diff(o) >= 0).all() and o[3] < o[4]               # -0 sorts just below +0: selection still returns a zero
    for x in v:
        assert ord2f(f2ord(np.array([x]))[0]) == x
