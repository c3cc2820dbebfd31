"""torch.distributed plumbing for multi-GPU runs: one process per GPU, no data-path collective.

The hot path does not exchange data between GPUs: whole grids are
replicated per rank (weak scaling) and the members of a batch (config 5's nearby trajectories,
PAPER.md:23) are independent, so they are sharded across ranks.  The only collectives are the
timing barrier, the max-over-ranks reduction of the device time and the final gather of results.
"""
from __future__ import annotations

import os

import numpy as np


def env_world() -> tuple[int, int, int]:
    """(rank, local_rank, world_size) from the torchrun environment (1 process if absent)."""
    return (int(os.environ.get("RANK", "0")), int(os.environ.get("LOCAL_RANK", "0")),
            int(os.environ.get("WORLD_SIZE", "1")))


def init(backend: str | None = None):
    """Initialise the default process group when launched under torchrun; returns (rank, world)."""
    import torch
    import torch.distributed as dist
    rank, local_rank, world = env_world()
    if world > 1 and not dist.is_initialized():
        if backend is None:
            backend = "nccl" if torch.cuda.is_available() else "gloo"
        os.environ.setdefault("MASTER_ADDR", "127.0.0.1")
        os.environ.setdefault("MASTER_PORT", "29500")
        if backend == "nccl":
            torch.cuda.set_device(local_rank)
            dist.init_process_group(backend, device_id=torch.device("cuda", local_rank))
        else:
            dist.init_process_group(backend)
    return rank, world


def barrier() -> None:
    import torch.distributed as dist
    if dist.is_available() and dist.is_initialized():
        dist.barrier()


def max_over_ranks(value: float) -> float:
    """Max of a host float over all ranks (the job's time is its slowest rank's)."""
    import torch
    import torch.distributed as dist
    if not (dist.is_available() and dist.is_initialized()):
        return float(value)
    dev = "cuda" if dist.get_backend() == "nccl" else "cpu"
    t = torch.tensor([float(value)], dtype=torch.float64, device=dev)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())


def sum_over_ranks(value: float) -> float:
    import torch
    import torch.distributed as dist
    if not (dist.is_available() and dist.is_initialized()):
        return float(value)
    dev = "cuda" if dist.get_backend() == "nccl" else "cpu"
    t = torch.tensor([float(value)], dtype=torch.float64, device=dev)
    dist.all_reduce(t, op=dist.ReduceOp.SUM)
    return float(t.item())


def shard_members(batch: int, rank: int, world: int) -> range:
    """Contiguous, balanced slice of batch members owned by `rank` (first ranks get the extras)."""
    if batch < 0 or world < 1 or not (0 <= rank < world):
        raise ValueError("bad shard arguments")
    base, extra = divmod(batch, world)
    lo = rank * base + min(rank, extra)
    return range(lo, lo + base + (1 if rank < extra else 0))


def shard_jvp_members(batch: int, rank: int, world: int) -> list[int]:
    """Members a rank integrates for the FD Jacobian-vector products: every rank needs the base
    trajectory (member 0) to form (phi(x + eps v_b) - phi(x))/eps locally, plus its share of the
    perturbed members 1..batch-1."""
    own = shard_members(batch - 1, rank, world)
    return [0] + [1 + b for b in own]


def gather_to_rank0(local: np.ndarray, counts: list[int]):
    """Concatenate per-rank arrays (leading dimension counts[r]) on rank 0; None elsewhere."""
    import torch
    import torch.distributed as dist
    if not (dist.is_available() and dist.is_initialized()):
        return local
    rank, world = dist.get_rank(), dist.get_world_size()
    dev = "cuda" if dist.get_backend() == "nccl" else "cpu"
    tail = local.shape[1:]
    pad = max(counts)
    buf = torch.zeros((pad,) + tail, dtype=torch.float64, device=dev)
    buf[: local.shape[0]] = torch.from_numpy(np.ascontiguousarray(local)).to(dev)
    out = [torch.empty_like(buf) for _ in range(world)] if rank == 0 else None
    dist.gather(buf, out, dst=0)
    if rank != 0:
        return None
    return np.concatenate([o[: counts[r]].cpu().numpy() for r, o in enumerate(out)], axis=0)
