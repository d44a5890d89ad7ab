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
