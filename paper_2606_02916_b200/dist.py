"""Multi-GPU plumbing: the path shards with NO data-path collective.

Rank r is the trainer of owner partition r % P (the paper's one-partition-per-node layout,
PAPER.md:251): its own partition's features sit in its HBM, every other partition in pinned
host memory, and it runs its own shard of the epoch's mini-batches through its own library
handle.  torch.distributed is used only for the barrier and the max/sum reductions of the
timing protocol (NCCL on GPUs, gloo in the CPU tests).
"""
from __future__ import annotations

import os
from typing import List, Sequence, Tuple

import torch
import torch.distributed as dist


def env_world() -> Tuple[int, int, int]:
    return (int(os.environ.get("RANK", "0")), int(os.environ.get("LOCAL_RANK", "0")),
            int(os.environ.get("WORLD_SIZE", "1")))


def init(backend: str) -> Tuple[int, int, int]:
    rank, local_rank, world = env_world()
    if world > 1 and not dist.is_initialized():
        os.environ.setdefault("MASTER_ADDR", "127.0.0.1")
        os.environ.setdefault("MASTER_PORT", "29500")
        dist.init_process_group(backend=backend, rank=rank, world_size=world)
    return rank, local_rank, world


def barrier():
    if dist.is_initialized():
        dist.barrier()


def _reduce(x: float, op, device) -> float:
    if not dist.is_initialized():
        return float(x)
    t = torch.tensor([x], dtype=torch.float64, device=device)
    dist.all_reduce(t, op=op)
    return float(t[0])


def max_over_ranks(x: float, device="cpu") -> float:
    return _reduce(x, dist.ReduceOp.MAX, device)


def sum_over_ranks(x: float, device="cpu") -> float:
    return _reduce(x, dist.ReduceOp.SUM, device)


def host_threads_for_rank(local_world_size: int = 0, hardware_threads: int = 0) -> int:
    """gg_config.host_threads for one of `local_world_size` ranks that share a host (default: the
    LOCAL_WORLD_SIZE torchrun exports).  One rank alone returns 0 = the library's default (0.4 x the
    hardware threads while copies are queued).  N ranks split that same budget -- the pack threads of all
    ranks read and write the one host DRAM that already bounds a single rank -- so each
    gets floor(0.4 x hardware threads / N), at least 1, as a hard cap."""
    n = local_world_size or int(os.environ.get("LOCAL_WORLD_SIZE", "1"))
    if n <= 1:
        return 0
    hw = hardware_threads or os.cpu_count() or 1
    budget = min(16, max(2, (hw * 2 + 2) // 5))
    return max(1, budget // n)


def shard_plan(rank: int, world: int, num_parts: int, n_batches: int) -> Tuple[int, List[int]]:
    """(local partition, batch indices) of a rank.  Replicated work, weak scaling: every rank is
    an independent trainer (of partition rank % P) that serves a full epoch's worth of batches in
    its OWN epoch order -- the generator's order rotated by the rank, so ranks see different
    windows.  The batch index that enters the sampling key (reading S7) is the position in that
    rank's order; with one rank the rotation is the identity.  This does not divide one epoch by N."""
    local_part = rank % num_parts
    shift = (rank * n_batches) // max(world, 1)
    order = [(i + shift) % n_batches for i in range(n_batches)]
    return local_part, order


def aggregate_throughput(units_this_rank: float, seconds_this_rank: float, device="cpu") -> Tuple[float, float]:
    """Whole-job throughput = units of all ranks / max over ranks of the time."""
    total = sum_over_ranks(units_this_rank, device)
    tmax = max_over_ranks(seconds_this_rank, device)
    return total / tmax, tmax
