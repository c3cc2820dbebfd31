"""Host-side multi-GPU plumbing (paper_1309_1720_b200/dist.py) on CPU: world_size 2, gloo.

The hot path has no data-path collective: batch members are sharded, every
rank integrates the base trajectory, results are gathered on rank 0.  Here the per-member "flow map"
is a cheap stand-in (the CUDA library needs a B200); what is tested is the sharding, the gather
order, the barrier and the max-over-ranks reduction that bench.py relies on.
"""
import os
import socket

import numpy as np
import pytest

from paper_1309_1720_b200 import dist as D


def test_shard_members_partition():
    for batch in (0, 1, 2, 5, 16, 17):
        for world in (1, 2, 3, 8):
            seen = []
            for r in range(world):
                seen += list(D.shard_members(batch, r, world))
            assert seen == list(range(batch))
            sizes = [len(D.shard_members(batch, r, world)) for r in range(world)]
            assert max(sizes) - min(sizes) <= 1
    with pytest.raises(ValueError):
        D.shard_members(4, 2, 2)


def test_shard_jvp_members_all_have_base():
    batch, world = 17, 4
    perturbed = []
    for r in range(world):
        m = D.shard_jvp_members(batch, r, world)
        assert m[0] == 0
        perturbed += m[1:]
    assert sorted(perturbed) == list(range(1, batch))


def _free_port() -> int:
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def _worker(rank: int, world: int, port: int, out_path: str):
    os.environ.update(RANK=str(rank), LOCAL_RANK=str(rank), WORLD_SIZE=str(world),
                      MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port))
    import torch.distributed as dist
    r, w = D.init("gloo")
    assert (r, w) == (rank, world)
    batch, eps = 7, 1e-7
    members = D.shard_jvp_members(batch, rank, world)
    # stand-in flow map: phi_b = b + 0.5 on a 2x3x4 "state"; J_b = (phi_b - phi_0)/eps
    phi = {b: np.full((2, 3, 4), b + 0.5) for b in members}
    local = np.stack([(phi[b] - phi[0]) / eps for b in members[1:]]) if len(members) > 1 \
        else np.zeros((0, 2, 3, 4))
    counts = [len(D.shard_members(batch - 1, q, world)) for q in range(world)]
    D.barrier()
    slowest = D.max_over_ranks(10.0 + rank)
    total = D.sum_over_ranks(1.0)
    J = D.gather_to_rank0(local, counts)
    if rank == 0:
        np.savez(out_path, J=J, slowest=slowest, total=total)
    else:
        assert J is None and slowest == 10.0 + world - 1
    dist.destroy_process_group()


def test_gloo_world2_shard_and_gather(tmp_path):
    import torch.multiprocessing as mp
    out = str(tmp_path / "rank0.npz")
    mp.spawn(_worker, args=(2, _free_port(), out), nprocs=2, join=True)
    got = np.load(out)
    assert got["slowest"] == 11.0 and got["total"] == 2.0
    J = got["J"]
    assert J.shape == (6, 2, 3, 4)
    for b in range(1, 7):
        assert np.allclose(J[b - 1], b / 1e-7, rtol=1e-12)


# ----------------------------------------------------------------------------- one grid over several ranks: row slabs
def test_slab_partition_and_ghosts():
    for ny, world, g, periodic in [(100, 3, 8, False), (64, 2, 4, True), (37, 4, 2, False), (512, 8, 8, True)]:
        slabs = [D.slab_of(ny, r, world, g, periodic) for r in range(world)]
        assert [s.lo for s in slabs] == [0] + [s.hi for s in slabs[:-1]] and slabs[-1].hi == ny
        for s in slabs:
            assert s.g_lo == (g if (periodic or s.rank > 0) else 0)
            assert s.g_hi == (g if (periodic or s.rank < world - 1) else 0)
            rows = s.global_rows()
            assert len(rows) == s.ext_rows and np.array_equal(rows[s.g_lo:s.g_lo + s.own], np.arange(s.lo, s.hi))
            # what a rank sends is exactly what its neighbour's ghost rows are images of
            if s.upper is not None:
                j0, n = s.send_to_upper()
                up = slabs[s.upper]
                k0, m = up.recv_from_lower()
                assert n == m == g and np.array_equal(rows[j0:j0 + n], up.global_rows()[k0:k0 + m])
            if s.lower is not None:
                j0, n = s.send_to_lower()
                lo = slabs[s.lower]
                k0, m = lo.recv_from_upper()
                assert n == m == g and np.array_equal(rows[j0:j0 + n], lo.global_rows()[k0:k0 + m])
    assert D.slab_of(50, 0, 1, 8, True).ext_rows == 50          # one rank: the context's own wrap is exact
    with pytest.raises(ValueError):
        D.slab_of(20, 0, 4, 8)                                   # 5-row slabs cannot feed 8 ghost rows
    assert D.ghost_depth(2, 4) == 8 and D.ghost_depth(1, 2, 3) == 6


class _OracleStepper:
    """Test stand-in for a cardiac.Context over an extended slab: the CPU oracle (test infrastructure)
    with the same step / get_rows / set_rows surface, CPU torch tensors as buffers."""

    def __init__(self, model, Z, dx, dt, scheme):
        self.model, self.Z, self.dx, self.dt, self.scheme = model, np.ascontiguousarray(Z), dx, dt, scheme

    def step(self, n):
        import oracle as O
        self.Z = O.step(self.model, self.Z, self.dx, self.dt, self.scheme, n)

    def get_rows(self, j0, n, dst=None):
        import torch
        t = torch.from_numpy(np.ascontiguousarray(self.Z[:, :, j0:j0 + n, :]))
        if dst is None:
            return t
        dst.copy_(t)
        return dst

    def set_rows(self, j0, src):
        self.Z[:, :, j0:j0 + src.shape[-2], :] = src.numpy()


def _slab_case(periodic):
    from paper_1309_1720_b200 import workloads as W
    cfg = W.make_config("slab", W.FHN, 24, W.LAP9X4, W.RK4, 0, batch=2, seed=4, ny=46,
                        boundary=1 if periodic else 0)
    return cfg, W.initial_state(cfg)


@pytest.mark.parametrize("periodic", [False, True])
@pytest.mark.parametrize("world,every", [(2, 1), (3, 1), (2, 2)])
def test_slabs_in_one_process_equal_the_single_grid_bitwise(world, every, periodic):
    """The decomposition argument itself, on the oracle: ghost depth r x substeps x k, one exchange per
    k steps, own rows bit for bit the undivided grid's (RK4, radius 2: 8 rows per step)."""
    import oracle as O
    cfg, Z = _slab_case(periodic)
    g = D.ghost_depth(2, 4, every)
    slabs = [D.slab_of(cfg.ny, r, world, g, periodic) for r in range(world)]
    steppers = [_OracleStepper(cfg.model, Z[:, :, s.global_rows(), :], cfg.dx, cfg.dt, cfg.scheme) for s in slabs]
    nsteps, left = 5, 5
    while left > 0:
        n = min(every, left)
        for st in steppers:
            st.step(n)
        left -= n
        if left > 0:
            D.exchange_local(steppers, slabs)
    got = np.concatenate([st.Z[:, :, s.g_lo:s.g_lo + s.own, :] for st, s in zip(steppers, slabs)], axis=2)
    ref = O.step(cfg.model, Z, cfg.dx, cfg.dt, cfg.scheme, nsteps)
    assert np.array_equal(got, ref)
    if every > 1:
        return
    # one ghost row too few and the cut shows (after one step; the trace a second step leaves 16 rows
    # away is below roundoff)
    slabs = [D.slab_of(cfg.ny, r, world, g - 1, periodic) for r in range(world)]
    steppers = [_OracleStepper(cfg.model, Z[:, :, s.global_rows(), :], cfg.dx, cfg.dt, cfg.scheme) for s in slabs]
    for st in steppers:
        st.step(every)
    bad = np.concatenate([st.Z[:, :, s.g_lo:s.g_lo + s.own, :] for st, s in zip(steppers, slabs)], axis=2)
    assert not np.array_equal(bad, O.step(cfg.model, Z, cfg.dx, cfg.dt, cfg.scheme, every))


def _slab_worker(rank: int, world: int, port: int, out_path: str, periodic: bool):
    os.environ.update(RANK=str(rank), LOCAL_RANK=str(rank), WORLD_SIZE=str(world),
                      MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port))
    import torch
    import torch.distributed as dist
    D.init("gloo")
    cfg, Z = _slab_case(periodic)
    slab = D.slab_of(cfg.ny, rank, world, D.ghost_depth(2, 4), periodic)
    st = _OracleStepper(cfg.model, Z[:, :, slab.global_rows(), :], cfg.dx, cfg.dt, cfg.scheme)
    alloc = lambda n: torch.empty((cfg.batch, cfg.n_v, n, cfg.nx), dtype=torch.float64)
    D.advance_slab(st, slab, 4, 1, lambda: D.exchange_dist(st, slab, alloc))
    full = D.gather_rows_to_rank0(st.Z[:, :, slab.g_lo:slab.g_lo + slab.own, :], cfg.ny)
    if rank == 0:
        np.save(out_path, full)
    else:
        assert full is None
    dist.destroy_process_group()


@pytest.mark.parametrize("periodic", [False, True])
def test_gloo_world2_slab_exchange(tmp_path, periodic):
    """exchange_dist over gloo, world size 2; with a periodic grid both neighbours of a rank are the
    same peer and the two messages are told apart by order and tag."""
    import torch.multiprocessing as mp
    import oracle as O
    out = str(tmp_path / "full.npy")
    mp.spawn(_slab_worker, args=(2, _free_port(), out, periodic), nprocs=2, join=True)
    cfg, Z = _slab_case(periodic)
    assert np.array_equal(np.load(out), O.step(cfg.model, Z, cfg.dx, cfg.dt, cfg.scheme, 4))
