"""World-size-2 `gloo` test of the host-side multi-GPU logic.

Plans are independent: the path shards over K with no data-path collective.  What the ranks share is
(1) the partition of the plan pool, (2) rank-dependent seeded weights in bench.py's weak-scaling mode,
(3) the max-over-ranks timing reduction.  The optimiser itself is stood in for by the oracle on a tiny case:
optimising a shard on its own must give the same plans as optimising the whole pool.
"""
import os
import sys
from pathlib import Path

import numpy as np
import pytest

ROOT = Path(__file__).resolve().parents[1]


def _worker(rank, world, port, tmp):
    sys.path.insert(0, str(ROOT))
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(world))
    import torch
    import torch.distributed as dist
    import bench
    import gmco_cases as gc
    import oracle
    dist.init_process_group("gloo", rank=rank, world_size=world)
    try:
        c = gc.make_case("C1", counts=(120, 40, 50, 50), n_plans=5)
        b, e = gc.shard_plans(c.n_plans, world, rank)
        r = oracle.optimize(c.D, c.structures, c.rx, c.T0, c.weights[b:e], m=5, iters=15)
        # gather of the per-rank results (the only exchange, after the loop): padded to the largest shard
        width = max(gc.shard_plans(c.n_plans, world, q)[1] - gc.shard_plans(c.n_plans, world, q)[0] for q in range(world))
        mine = torch.zeros(width, dtype=torch.float64); mine[: e - b] = torch.from_numpy(r["F"])
        parts = [torch.zeros(width, dtype=torch.float64) for _ in range(world)]
        dist.all_gather(parts, mine)
        F = np.concatenate([parts[q][: np.diff(gc.shard_plans(c.n_plans, world, q))[0]].numpy() for q in range(world)])
        # timing reduction: the slowest rank decides
        ms = bench.max_over_ranks_ms(10.0 + 5.0 * rank, world, "cpu")
        # weak-scaling mode: every rank draws its own pool from seed 7 + rank
        w_own = gc.make_case("C1", counts=(120, 40, 50, 50), n_plans=3, seed_weights=7 + rank).weights
        ws = [torch.zeros(w_own.shape, dtype=torch.float32) for _ in range(world)]
        dist.all_gather(ws, torch.from_numpy(w_own))
        if rank == 0:
            np.savez(tmp, F=F, ms=ms, w0=ws[0].numpy(), w1=ws[1].numpy())
    finally:
        dist.destroy_process_group()


def test_k_sharding_over_two_ranks(tmp_path):
    import torch.multiprocessing as mp
    import gmco_cases as gc
    import oracle
    import bench
    oracle.build()
    out = str(tmp_path / "gloo.npz")
    port = 29500 + os.getpid() % 2000
    mp.spawn(_worker, args=(2, port, out), nprocs=2, join=True)
    z = np.load(out)
    c = gc.make_case("C1", counts=(120, 40, 50, 50), n_plans=5)
    whole = oracle.optimize(c.D, c.structures, c.rx, c.T0, c.weights, m=5, iters=15)["F"]
    assert np.array_equal(z["F"], whole)                 # a plan does not depend on which shard it is in
    assert float(z["ms"]) == 15.0                        # max over ranks
    assert not np.array_equal(z["w0"], z["w1"])          # different pools per rank
    assert bench.job_value(1000, 2, 5, 100.0) == pytest.approx(2 * 1000 * 5 / 0.1)
