"""Event sharding across ranks: host logic only, no arithmetic of the method.

Events are independent and the RNG is keyed by the GLOBAL event index, so rank g of G takes a contiguous index
range and produces bit-identical events to a single-GPU run: there is no data-path collective during generation.
Unweighting needs (1) w_max, which every rank obtains by replaying the same pre-run events 0..prerun-1
(deterministic, zero communication), and (2) for a globally ordered compacted list, the exclusive scan of the
per-rank accepted counts: one all_gather of an int64 per rank.
"""
from __future__ import annotations

from typing import List, Tuple


def shard_range(n_events: int, rank: int, world: int) -> Tuple[int, int]:
    """(event_offset, count) of `rank`: contiguous, ordered by rank, sizes differ by at most one (strong scaling)."""
    if not (0 <= rank < world) or n_events < 0:
        raise ValueError("bad shard request")
    base, rem = divmod(n_events, world)
    count = base + (1 if rank < rem else 0)
    offset = rank * base + min(rank, rem)
    return offset, count


def weak_range(n_per_rank: int, rank: int) -> Tuple[int, int]:
    """(event_offset, count) with a fixed per-rank batch (weak scaling): rank g owns [g*n, (g+1)*n)."""
    return rank * n_per_rank, n_per_rank


def output_offsets(counts: List[int]) -> List[int]:
    """Exclusive scan of the per-rank accepted counts = where each rank's compacted events start globally."""
    out, acc = [], 0
    for c in counts:
        out.append(acc)
        acc += int(c)
    return out


def gather_counts(local_count: int, group=None) -> List[int]:
    """all_gather of one int64 per rank (NCCL on GPUs, gloo in the CPU tests); single process -> [local_count]."""
    import torch
    import torch.distributed as dist
    if not (dist.is_available() and dist.is_initialized()):
        return [int(local_count)]
    backend = dist.get_backend(group)
    dev = torch.device("cuda", torch.cuda.current_device()) if backend == "nccl" else torch.device("cpu")
    mine = torch.tensor([int(local_count)], dtype=torch.int64, device=dev)
    world = dist.get_world_size(group)
    buf = [torch.zeros_like(mine) for _ in range(world)]
    dist.all_gather(buf, mine, group=group)
    return [int(b.item()) for b in buf]
