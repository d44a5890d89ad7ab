"""Multi-process plumbing for bench.py (one process per GPU, torch.distributed).

The causal-set action path runs on one GPU and does not shard (BASELINE.json
north_star): with N ranks every rank runs
an independent replica (its own seeded sprinkling) and there is no data-path
collective.  Only the measurement is reduced: elapsed time as the MAX over
ranks, processed units as the SUM.  The same code runs over `gloo` on CPU
(tests/test_dist_gloo.py) and `nccl` on GPUs.
"""
from __future__ import annotations

import os

import torch
import torch.distributed as dist


def env_world():
    """(rank, local_rank, world_size) from the torchrun environment (1 process if absent)."""
    return (int(os.environ.get("RANK", "0")), int(os.environ.get("LOCAL_RANK", "0")),
            int(os.environ.get("WORLD_SIZE", "1")))


def init(backend: str | None = None):
    rank, local_rank, world = env_world()
    if world > 1 and not dist.is_initialized():
        os.environ.setdefault("MASTER_ADDR", "127.0.0.1")
        os.environ.setdefault("MASTER_PORT", "29500")
        if backend is None:
            backend = "nccl" if torch.cuda.is_available() else "gloo"
        dist.init_process_group(backend=backend, rank=rank, world_size=world)
    return rank, local_rank, world


def barrier():
    if dist.is_initialized():
        dist.barrier()


def _device():
    if dist.is_initialized() and dist.get_backend() == "nccl":
        return torch.device("cuda", torch.cuda.current_device())
    return torch.device("cpu")


def reduce_max(x: float) -> float:
    if not dist.is_initialized():
        return float(x)
    t = torch.tensor([x], dtype=torch.float64, device=_device())
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())


def reduce_sum(x: float) -> float:
    if not dist.is_initialized():
        return float(x)
    t = torch.tensor([x], dtype=torch.float64, device=_device())
    dist.all_reduce(t, op=dist.ReduceOp.SUM)
    return float(t.item())


def all_reduce_sum_(t: torch.Tensor) -> torch.Tensor:
    """In-place sum over ranks of an integer tensor (the partial interval histograms of `shard_rows`): NCCL when
    the tensor is on a GPU, gloo on the CPU; a no-op with one process."""
    if dist.is_initialized() and dist.get_world_size() > 1:
        dist.all_reduce(t, op=dist.ReduceOp.SUM)
    return t


def shard_rows(N: int, world: int, tile: int = 256):
    """Contiguous row ranges [(begin, end)] * world of the outer element i of a2, cut on tile borders so that every
    rank gets about the same tensor work (NEXT-4; the paper splits row groups over MPI ranks).
    Row tile I of nT pairs with the tiles J >= I, tile (I, J) costing J - I + 1 K stages, so tile I costs
    (nT - I)(nT - I + 1) / 2: early rows are far more expensive than late ones.  Greedy prefix cut at k/world of
    the total; ranks beyond the number of tiles get empty ranges.  Pure host arithmetic."""
    nT = (N + tile - 1) // tile
    cost = [(nT - I) * (nT - I + 1) // 2 for I in range(nT)]
    total = sum(cost)
    cuts, acc, I = [0], 0, 0
    for r in range(1, world):
        target = total * r / world
        while I < nT and acc + cost[I] / 2 <= target:
            acc += cost[I]
            I += 1
        cuts.append(I)
    cuts.append(nT)
    return [(min(N, cuts[r] * tile), min(N, cuts[r + 1] * tile)) for r in range(world)]


def replica_seed(base_seed: int, rank: int) -> int:
    """Replica `rank` sprinkles with its own seed (rank 0 keeps the config's seed)."""
    return base_seed + 1000003 * rank


def aggregate(units_this_rank: float, seconds_this_rank: float):
    """Whole-job throughput: sum of units over ranks / max of elapsed time over ranks."""
    units = reduce_sum(units_this_rank)
    secs = reduce_max(seconds_this_rank)
    return units, secs, (units / secs if secs > 0 else 0.0)


def shutdown():
    if dist.is_initialized():
        dist.destroy_process_group()
