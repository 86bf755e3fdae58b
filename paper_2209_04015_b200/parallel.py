"""Host-side helpers for running the library on several GPUs of one node (one process per GPU).

The path shards over walkers only ("walkers per task"): every rank holds a replica of the
half-rotated tensors and evaluates its own walkers with ``LocalEnergy``; there is no collective on the data path.
What is left for the host is bookkeeping: which walkers a rank owns, gathering the per-walker results, and taking
the maximum of a timing over ranks.  Everything here works with any ``torch.distributed`` backend (``nccl`` on GPUs,
``gloo`` in the CPU tests).
"""
from __future__ import annotations

import torch
import torch.distributed as dist


def walker_shard(n_walkers: int, rank: int, world: int) -> tuple[int, int]:
    """(start, count) of the contiguous walker block owned by ``rank``: the first ``n_walkers % world`` ranks get
    one walker more.  Counts may be zero when there are fewer walkers than ranks."""
    if not (0 <= rank < world) or n_walkers < 0:
        raise ValueError("walker_shard: need 0 <= rank < world and n_walkers >= 0")
    base, rem = divmod(n_walkers, world)
    count = base + (1 if rank < rem else 0)
    start = rank * base + min(rank, rem)
    return start, count


def gather_walker_results(local: torch.Tensor, n_walkers: int, group=None) -> torch.Tensor:
    """All-gather per-walker complex128 results (energies or log-overlaps) of every rank's shard into the global
    walker order.  ``local`` holds this rank's ``walker_shard`` block.  One collective of ``n_walkers`` complex
    numbers; shards are padded to the largest count so that ranks with uneven shards can take part."""
    world = dist.get_world_size(group) if dist.is_initialized() else 1
    rank = dist.get_rank(group) if dist.is_initialized() else 0
    start, count = walker_shard(n_walkers, rank, world)
    if local.numel() != count:
        raise ValueError(f"gather_walker_results: rank {rank} passed {local.numel()} values, owns {count}")
    if world == 1:
        return local.clone()
    maxc = -(-n_walkers // world)
    buf = torch.zeros(2 * maxc, dtype=torch.float64, device=local.device)
    buf[: 2 * count] = torch.view_as_real(local.to(torch.complex128)).reshape(-1)
    parts = [torch.empty_like(buf) for _ in range(world)]
    dist.all_gather(parts, buf, group=group)
    out = torch.empty(n_walkers, dtype=torch.complex128, device=local.device)
    for r in range(world):
        s, c = walker_shard(n_walkers, r, world)
        out[s:s + c] = torch.view_as_complex(parts[r][: 2 * c].reshape(c, 2))
    return out


def max_over_ranks(value: float, device=None, group=None) -> float:
    """Maximum of a host scalar (a device-measured time) over all ranks."""
    if not dist.is_initialized() or dist.get_world_size(group) == 1:
        return float(value)
    t = torch.tensor([float(value)], dtype=torch.float64, device=device)
    dist.all_reduce(t, op=dist.ReduceOp.MAX, group=group)
    return float(t.item())
