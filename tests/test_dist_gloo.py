"""world_size-2 gloo test of the N>1 measurement path used by bench.py (replicas only)."""
import os
import socket

import pytest
import torch
import torch.multiprocessing as mp


def _free_port():
    s = socket.socket()
    s.bind(("127.0.0.1", 0))
    p = s.getsockname()[1]
    s.close()
    return p


def _worker(rank, world, port, out_dir):
    os.environ.update(RANK=str(rank), LOCAL_RANK=str(rank), WORLD_SIZE=str(world),
                      MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port))
    from paper_1805_04463_b200 import dist as csd, inputs as inp
    r, lr, w = csd.init(backend="gloo")
    assert (r, w) == (rank, world)
    csd.barrier()
    # every rank: its own replica; rank-dependent units and time
    seed = csd.replica_seed(inp.CONFIGS[1].seed, rank)
    coords = inp.sprinkle(inp.GEOM_MINK2_LIGHTCONE, 2, 64, seed)
    units, secs, thr = csd.aggregate(100.0 * (rank + 1), 0.5 * (rank + 1))
    with open(os.path.join(out_dir, "r%d.txt" % rank), "w") as f:
        f.write("%r %r %r %r\n" % (units, secs, thr, float(coords.sum())))
    csd.barrier()
    csd.shutdown()


def test_two_rank_aggregation(tmp_path):
    port = _free_port()
    mp.spawn(_worker, args=(2, port, str(tmp_path)), nprocs=2, join=True)
    rows = [open(tmp_path / ("r%d.txt" % r)).read().split() for r in range(2)]
    for row in rows:
        assert float(row[0]) == 300.0          # sum of units
        assert float(row[1]) == 1.0            # max of times
        assert float(row[2]) == 300.0
    assert rows[0][3] != rows[1][3]            # replicas sprinkle different causets


def test_single_process_passthrough():
    from paper_1805_04463_b200 import dist as csd
    assert csd.aggregate(10.0, 2.0) == (10.0, 2.0, 5.0)
    assert csd.replica_seed(7, 0) == 7


# ---- NEXT-4: rows of one causet split over the ranks + one all-reduce of the histogram ----------------
def test_shard_rows_partition():
    """Host arithmetic of the row split: the ranges tile [0, N) in order on 256-row borders, and no rank carries
    much more than its share of the tensor work (tile I costs (nT - I)(nT - I + 1) / 2 stages)."""
    from paper_1805_04463_b200 import dist as csd
    for N in (1, 255, 256, 1000, 16384, 65536, 131072, 100001):
        for world in (1, 2, 3, 4, 8):
            parts = csd.shard_rows(N, world)
            assert len(parts) == world and parts[0][0] == 0 and parts[-1][1] == N
            for (a, b), (c, d) in zip(parts, parts[1:]):
                assert a <= b == c <= d
            assert all(a % 256 == 0 for a, _ in parts if a < N)
            nT = (N + 255) // 256
            cost = lambda a, b: sum((nT - I) * (nT - I + 1) // 2 for I in range(a // 256, (b + 255) // 256))
            total = cost(0, N)
            if nT >= 16 * world:
                assert max(cost(a, b) for a, b in parts) <= 1.15 * total / world


def _shard_worker(rank, world, port, out_dir):
    os.environ.update(RANK=str(rank), LOCAL_RANK=str(rank), WORLD_SIZE=str(world),
                      MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port))
    import numpy as np
    import oracle
    from paper_1805_04463_b200 import dist as csd, inputs as inp
    csd.init(backend="gloo")
    cfg = inp.CONFIGS[3]
    N = 3000
    coords = inp.make_config_coords(cfg, N=N)          # every rank: the same causet
    bits = oracle.causal_matrix_bits(coords, cfg.geometry)
    r0, r1 = csd.shard_rows(N, world)[rank]
    part = oracle.interval_hist_alg20(bits, N, r0, r1)[0]      # stands in for cs_interval_hist_ex(row range)
    total = csd.all_reduce_sum_(torch.from_numpy(part.copy()))
    np.save(os.path.join(out_dir, "h%d.npy" % rank), total.numpy())
    csd.barrier()
    csd.shutdown()


def test_two_rank_row_sharding_sums_to_the_whole_histogram(tmp_path):
    """bench.py --shard's plumbing at world size 2 over gloo: partial histograms of disjoint row ranges, one
    all-reduce(sum), every rank ends with the single-process histogram (bit-exact)."""
    import numpy as np
    import oracle
    from paper_1805_04463_b200 import inputs as inp
    port = _free_port()
    mp.spawn(_shard_worker, args=(2, port, str(tmp_path)), nprocs=2, join=True)
    cfg = inp.CONFIGS[3]
    coords = inp.make_config_coords(cfg, N=3000)
    want = oracle.interval_hist_alg20(oracle.causal_matrix_bits(coords, cfg.geometry), 3000)[0]
    for r in range(2):
        assert np.array_equal(np.load(tmp_path / ("h%d.npy" % r)), want)
