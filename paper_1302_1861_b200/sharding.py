"""Multi-GPU plumbing of the hot path: one process per GPU, records sharded by
contiguous load-order ranges, no collective in the data path.

Records are independent and the paper itself spreads a job over GPUs as replicas that draw
different particles, so every rank builds its own counts / offsets / batches from its own
shard.  The only exchange the method can ever need is the one below: if a consumer wants globally contiguous
slots, the ranks all-gather ``counts[K]`` (<= 4.9 MB) and take a per-key exclusive prefix over ranks --
particles never move.  ``torch.distributed`` is the transport (NCCL on GPUs, gloo in the CPU tests).
"""
from __future__ import annotations

from typing import Tuple

import torch
import torch.distributed as dist


def shard_range(rank: int, world: int, n_total: int) -> Tuple[int, int]:
    """(first record, number of records) of ``rank``: contiguous, multiples of 4 records except the last shard
    (psl_load_chunk wants every chunk but the last to be a multiple of 4)."""
    per = -(-n_total // world)
    per += (-per) % 4
    first = min(rank * per, n_total)
    return first, min(per, n_total - first)


def global_offsets(local_counts: torch.Tensor, group=None) -> Tuple[torch.Tensor, torch.Tensor]:
    """Slots of this rank's buckets in the rank-major-within-key global order.

    local_counts: counts[K] of this rank (any integer dtype, CPU or CUDA).  Returns (first_slot[K], total[K]):
    first_slot[k] = sum of all ranks' counts of keys < k + counts[k] of the ranks before this one, so that
    key k of the whole job is one contiguous run ordered by (rank, local order) = global load order when
    shards are contiguous ranges.  total[k] = count of key k over all ranks."""
    world = dist.get_world_size(group)
    rank = dist.get_rank(group)
    c = local_counts.to(torch.int64)
    gathered = [torch.empty_like(c) for _ in range(world)]
    dist.all_gather(gathered, c, group=group)
    allc = torch.stack(gathered)                       # [world, K]
    total = allc.sum(dim=0)
    key_start = torch.cumsum(total, dim=0) - total     # exclusive prefix over keys
    before = allc[:rank].sum(dim=0) if rank > 0 else torch.zeros_like(total)
    return key_start + before, total


def max_over_ranks(ms: float, device=None, group=None) -> float:
    """The slowest rank defines the job (bench.py's timing rule)."""
    t = torch.tensor([ms], dtype=torch.float64, device=device)
    dist.all_reduce(t, op=dist.ReduceOp.MAX, group=group)
    return float(t.item())
