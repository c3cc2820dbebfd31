"""torch.distributed plumbing for multi-GPU runs: one process per GPU.

The BASELINE configs do not exchange data between GPUs: whole grids are
replicated per rank (weak scaling) and the members of a batch (config 5's nearby trajectories,
PAPER.md:23) are independent, so they are sharded across ranks; the only collectives there are the
timing barrier, the max-over-ranks reduction of the device time and the final gather of results.
ONE grid larger than a GPU should carry is cut into row slabs (second half of this file): the only
point-to-point exchange of the package, one ghost-row message per neighbour every k time steps.
"""
from __future__ import annotations

import dataclasses
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


# ----------------------------------------------------------------------------- ONE grid over several GPUs: row slabs
# SURVEY.md 8(e) / f4.  A single grid does not shard without communication: every substep reads r rows
# across each cut ("lock-step").  Exchanging after every substep would cost a message
# latency per substep; instead a rank keeps g = r x substeps x k ghost rows towards each neighbour and
# advances its EXTENDED slab k whole time steps with the unchanged single-GPU kernels.  Information
# travels r rows per substep, so whatever the artificial edge of the extended slab does, it reaches
# ghost rows only: the rank's own rows are bit for bit the single-grid result, and ONE exchange per k
# time steps refreshes the ghosts (cardiac_get_rows on the sender, cardiac_set_rows on the receiver;
# NCCL send/recv over NVLink in between, or a peer-mapped destination for cardiac_get_rows).


def ghost_depth(radius: int, substeps: int, steps_between_exchanges: int = 1) -> int:
    """Ghost rows per cut: r rows per substep, `substeps` per time step."""
    if radius < 1 or substeps < 1 or steps_between_exchanges < 1:
        raise ValueError("bad ghost arguments")
    return radius * substeps * steps_between_exchanges


@dataclasses.dataclass(frozen=True)
class Slab:
    """Rows [lo, hi) of a grid of ny rows owned by `rank`, held with g_lo ghost rows below lo and g_hi
    above hi - 1 (0 at a physical no-flux edge, where the context's own boundary rule is the real one)."""
    rank: int
    world: int
    ny: int
    lo: int
    hi: int
    g_lo: int
    g_hi: int
    periodic: bool

    @property
    def own(self) -> int:
        return self.hi - self.lo

    @property
    def ext_rows(self) -> int:
        return self.g_lo + self.own + self.g_hi

    @property
    def lower(self):
        """Rank that owns the rows below lo (None at a physical edge)."""
        if self.g_lo == 0:
            return None
        return (self.rank - 1) % self.world

    @property
    def upper(self):
        if self.g_hi == 0:
            return None
        return (self.rank + 1) % self.world

    def global_rows(self) -> np.ndarray:
        """Global row index of every row of the extended slab (wrapped for a periodic grid)."""
        return np.arange(self.lo - self.g_lo, self.hi + self.g_hi) % self.ny

    # rows of the EXTENDED slab (local indices) that an exchange reads and writes
    def send_to_lower(self) -> tuple[int, int]:   # my lowest own rows -> the lower rank's upper ghosts
        return self.g_lo, self.g_lo
    def send_to_upper(self) -> tuple[int, int]:   # my highest own rows -> the upper rank's lower ghosts
        return self.g_lo + self.own - self.g_hi, self.g_hi
    def recv_from_lower(self) -> tuple[int, int]:
        return 0, self.g_lo
    def recv_from_upper(self) -> tuple[int, int]:
        return self.g_lo + self.own, self.g_hi


def slab_of(ny: int, rank: int, world: int, ghost: int, periodic: bool = False) -> Slab:
    """Balanced contiguous row slab of `rank` with `ghost` rows towards each neighbouring rank."""
    rows = shard_members(ny, rank, world)
    if world == 1:
        return Slab(rank, world, ny, 0, ny, 0, 0, periodic)   # the context's own boundary rule is exact
    if min(len(shard_members(ny, r, world)) for r in range(world)) < ghost:
        raise ValueError(f"slabs of {ny} rows over {world} ranks are thinner than the {ghost} ghost rows")
    g_lo = ghost if (periodic or rank > 0) else 0
    g_hi = ghost if (periodic or rank < world - 1) else 0
    return Slab(rank, world, ny, rows.start, rows.stop, g_lo, g_hi, periodic)


def exchange_local(steppers, slabs) -> None:
    """Ghost refresh between slabs that live in ONE process (several contexts on one GPU, or one per
    visible device): rows go straight from get_rows to set_rows.  `steppers[r]` serves `slabs[r]`."""
    sends = {}
    for st, sl in zip(steppers, slabs):
        if sl.lower is not None:
            sends[(sl.rank, "down")] = st.get_rows(*sl.send_to_lower())
        if sl.upper is not None:
            sends[(sl.rank, "up")] = st.get_rows(*sl.send_to_upper())
    for st, sl in zip(steppers, slabs):
        if sl.lower is not None:
            st.set_rows(sl.recv_from_lower()[0], sends[(sl.lower, "up")])
        if sl.upper is not None:
            st.set_rows(sl.recv_from_upper()[0], sends[(sl.upper, "down")])


def exchange_dist(stepper, slab: Slab, alloc) -> None:
    """Ghost refresh across ranks: 2 sends + 2 receives per rank in one batch (NCCL groups them;
    gloo matches by tag).  `alloc(nrows)` returns an empty dense [batch][n_v][nrows][nx] float64 tensor
    on the backend's device; stepper.get_rows(j0, n, dst) / set_rows(j0, src) are the C-ABI calls."""
    import torch.distributed as dist
    ops, recvs = [], []
    TAG_DOWN, TAG_UP = 1, 2      # direction the rows travel
    if slab.lower is not None:
        j0, n = slab.send_to_lower()
        ops.append(dist.P2POp(dist.isend, stepper.get_rows(j0, n, alloc(n)), slab.lower, tag=TAG_DOWN))
    if slab.upper is not None:
        j0, n = slab.send_to_upper()
        ops.append(dist.P2POp(dist.isend, stepper.get_rows(j0, n, alloc(n)), slab.upper, tag=TAG_UP))
    # receive order mirrors the peers' send order (the k-th send to a peer meets its k-th receive):
    # the upper rank's first send travels down, into my upper ghosts
    if slab.upper is not None:
        j0, n = slab.recv_from_upper()
        buf = alloc(n)
        ops.append(dist.P2POp(dist.irecv, buf, slab.upper, tag=TAG_DOWN))
        recvs.append((j0, buf))
    if slab.lower is not None:
        j0, n = slab.recv_from_lower()
        buf = alloc(n)
        ops.append(dist.P2POp(dist.irecv, buf, slab.lower, tag=TAG_UP))
        recvs.append((j0, buf))
    if not ops:
        return
    for req in dist.batch_isend_irecv(ops):
        req.wait()
    for j0, buf in recvs:
        stepper.set_rows(j0, buf)


def advance_slab(stepper, slab: Slab, nsteps: int, every: int, exchange) -> None:
    """nsteps time steps of the extended slab, ghosts refreshed every `every` steps by exchange()."""
    left = nsteps
    while left > 0:
        n = min(every, left)
        stepper.step(n)
        left -= n
        if left > 0:
            exchange()


def gather_rows_to_rank0(own: np.ndarray, ny: int):
    """Own rows [batch][n_v][rows][nx] of every rank -> the full [batch][n_v][ny][nx] on rank 0."""
    import torch.distributed as dist
    world = dist.get_world_size() if (dist.is_available() and dist.is_initialized()) else 1
    counts = [len(shard_members(ny, r, world)) for r in range(world)]
    rows_first = np.ascontiguousarray(np.moveaxis(own, 2, 0))
    full = gather_to_rank0(rows_first, counts)
    return None if full is None else np.ascontiguousarray(np.moveaxis(full, 0, 2))
