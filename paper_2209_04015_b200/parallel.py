"""Host-side helpers for running the library on several GPUs of one node (one process per GPU).

The path shards over walkers only ("walkers per task"): every rank holds a replica of the
half-rotated tensors and evaluates its own walkers with ``LocalEnergy``; there is no collective on the data path.
What is left for the host is bookkeeping: which walkers a rank owns, gathering the per-walker results, and taking
the maximum of a timing over ranks.  Everything here works with any ``torch.distributed`` backend (``nccl`` on GPUs,
``gloo`` in the CPU tests).
"""
from __future__ import annotations

import hashlib
import os
import socket
import subprocess
import sys

import torch
import torch.distributed as dist


def torchrun_command(script: str, nproc: int, argv: list[str], port: int | None = None) -> list[str]:
    """The command line that runs ``script argv`` as ``nproc`` ranks on this node (one process per GPU), the way
    the benchmark driver launches it: ``python -m torch.distributed.run --nnodes=1 --nproc-per-node N ...``."""
    if port is None:
        with socket.socket() as s:
            s.bind(("127.0.0.1", 0))
            port = s.getsockname()[1]
    return [sys.executable, "-m", "torch.distributed.run", "--nnodes=1", f"--nproc-per-node={nproc}",
            "--master-addr", "127.0.0.1", "--master-port", str(port), script, *argv]


def respawn_under_torchrun(script: str, nproc: int, argv: list[str], **popen_kw) -> subprocess.CompletedProcess:
    """Re-run ``script`` as ``nproc`` ranks (used when a multi-rank run was asked for from a plain ``python`` call,
    i.e. WORLD_SIZE is not set).  Returns the finished process; stdout/stderr pass through unless redirected."""
    env = dict(os.environ)
    env.pop("RANK", None)
    env.pop("LOCAL_RANK", None)
    return subprocess.run(torchrun_command(script, nproc, argv), env=env, **popen_kw)


def init_from_env(backend: str, device=None) -> tuple[int, int, int]:
    """(rank, world, local_rank) from the torchrun environment; initialises the process group when world > 1."""
    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    local_rank = int(os.environ.get("LOCAL_RANK", "0"))
    if world > 1 and not dist.is_initialized():
        os.environ.setdefault("MASTER_ADDR", "127.0.0.1")
        if device is not None:
            dist.init_process_group(backend, device_id=device)
        else:
            dist.init_process_group(backend)
    return rank, world, local_rank


def weak_scaling_block(walkers_per_rank: int, rank: int, world: int) -> tuple[int, int]:
    """Weak scaling: the job has ``world * walkers_per_rank`` walkers and rank r owns the r-th block of them (the
    ``walker_shard`` of the global population), so the first block is exactly the one-rank job's population."""
    return walker_shard(world * walkers_per_rank, rank, world)


def result_digest(values: torch.Tensor) -> str:
    """SHA-256 of the raw bytes of per-walker complex128 results: equal digests mean bit-identical results."""
    v = values.detach().to("cpu", torch.complex128).contiguous()
    return hashlib.sha256(torch.view_as_real(v).numpy().tobytes()).hexdigest()


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
