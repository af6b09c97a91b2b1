"""Host-side model of the compaction index scheme.  The tensor kernels re-deal a FIXED grid of CTAs
over the plan tiles that still hold running plans (`compact_remap`, `compact_remap_pair` in csrc/kernels_tc.cu) and
`k_step` derives, from the running count alone, which partial-sum slots belong to a plan's tile (`reduce_partials` in
csrc/kernels_lbfgs.cu).  The three must agree.  This file restates the integer formulas and checks the properties the
design relies on for every grid the library can launch: each (active tile, segment) is owned by exactly one CTA (or CTA
pair), slots stay inside the buffers sized by gmco_api.cu (tiles x segs), the reader's slot range is exactly what the
writers of that tile wrote, and the point segments tile [0, n_chunks) without gaps.  It does not run the kernels; the
-m gpu parity tests do."""
import itertools

import pytest


def remap_single(gx, gy, bx, by, n_running, cap):
    """compact_remap: grid (segs, tiles) = (gx, gy)."""
    ta = (n_running + 127) >> 7
    total = gx * gy
    sa = min(total // ta, cap)
    c = by * gx + bx
    tile = c // sa
    return (tile < ta), tile, c - tile * sa, sa


def remap_pair(gx, gy, bx, by, n_running, cap):
    """compact_remap_pair: grid (tiles, segs) = (gx, gy), cluster (2, 1, 1); rank = bx & 1."""
    rank = bx & 1
    tap = (((n_running + 127) >> 7) + 1) >> 1
    total = gy * (gx >> 1)
    sa = min(total // tap, cap)
    c = by * (gx >> 1) + (bx >> 1)
    pt = c // sa
    return (pt < tap), 2 * pt + rank, c - pt * sa, sa


def reader_range(total_ctas, cap, n_running, row, pair, grad_pair=False):
    """reduce_partials: slot range [f0, f1) of the objective partials and [g0, g1) of the gradient partials
    (grad_pair: k_grad_tc_pair deals its CTA pairs like the dose pair kernel, gmco_options.dose_kernel = 2)."""
    ta = (n_running + 127) >> 7
    sa = min(total_ctas // ta, cap)
    g0 = (row >> 7) * sa
    g = (g0, g0 + sa)
    if pair:
        sa = min((total_ctas >> 1) // ((ta + 1) >> 1), cap)
    f0 = (row >> 7) * sa
    if grad_pair:
        g = (f0, f0 + sa)
    return (f0, f0 + sa), g


GRIDS = [(1, 148), (2, 74), (3, 49), (4, 37), (8, 18), (16, 9), (32, 9), (32, 4), (79, 5), (80, 1)]     # (tiles, segs)


@pytest.mark.parametrize("tiles,segs", GRIDS)
def test_single_cta_remap_covers_each_active_tile_segment_once(tiles, segs):
    cap = max(segs, 36)
    for n_running in sorted(n for n in {1, 2, 127, 128, 129, 128 * tiles - 1, 128 * tiles} | set(range(1, 128 * tiles + 1, 97)) if n <= 128 * tiles):
        ta = (n_running + 127) >> 7
        owners = {}
        for by, bx in itertools.product(range(tiles), range(segs)):
            ok, tile, seg, sa = remap_single(segs, tiles, bx, by, n_running, cap)
            if not ok:
                continue
            assert 0 <= seg < sa and tile < ta
            assert (tile, seg) not in owners
            owners[(tile, seg)] = (bx, by)
            assert tile * sa + seg < tiles * segs                      # Fpart / Gpart slot inside the buffer
        assert len(owners) == ta * sa                                   # every (active tile, segment) has its CTA
        for row in range(0, n_running, 61):
            f, g = reader_range(tiles * segs, cap, n_running, row, pair=False)
            written = sorted(t * sa + s for (t, s) in owners if t == row >> 7)
            assert written == list(range(*g)) == list(range(*f))


@pytest.mark.parametrize("tiles,segs", [g for g in GRIDS if g[0] % 2 == 0])
def test_pair_remap_keeps_pairs_together_and_matches_the_reader(tiles, segs):
    cap = max(segs, 36)
    for n_running in sorted(n for n in {1, 128, 129, 256, 257, 128 * tiles} | set(range(1, 128 * tiles + 1, 113)) if n <= 128 * tiles):
        ta = (n_running + 127) >> 7
        owners = {}
        for by, bx in itertools.product(range(segs), range(tiles)):
            ok, tile, seg, sa = remap_pair(tiles, segs, bx, by, n_running, cap)
            ok2, tile2, seg2, _ = remap_pair(tiles, segs, bx ^ 1, by, n_running, cap)
            assert ok == ok2 and seg == seg2 and tile ^ 1 == tile2       # the two CTAs of a cluster never part
            if not ok:
                continue
            assert (tile, seg) not in owners
            owners[(tile, seg)] = (bx, by)
            assert tile < tiles and tile * sa + seg < tiles * segs
        for t in range(ta):                                             # every active tile has all its segments
            assert sorted(s for (tt, s) in owners if tt == t) == list(range(sa))
        for row in range(0, n_running, 53):
            f, _ = reader_range(tiles * segs, cap, n_running, row, pair=True)
            assert sorted(t * sa + s for (t, s) in owners if t == row >> 7) == list(range(*f))
            f2, g2 = reader_range(tiles * segs, cap, n_running, row, pair=True, grad_pair=True)
            assert f2 == f and g2 == f                                   # the pair gradient kernel writes the same slots


@pytest.mark.parametrize("n_chunks,segs", [(12, 148), (94, 18), (94, 36), (94, 5), (313, 9), (47, 74), (1, 3)])
def test_point_segments_tile_the_chunks(n_chunks, segs):
    """c0 = seg n / segs, c1 = (seg + 1) n / segs: contiguous, complete, at most one chunk apart in length."""
    edges = [(s * n_chunks) // segs for s in range(segs + 1)]
    assert edges[0] == 0 and edges[-1] == n_chunks and all(b >= a for a, b in zip(edges, edges[1:]))
    lens = [b - a for a, b in zip(edges, edges[1:])]
    assert max(lens) - min(lens) <= 1
