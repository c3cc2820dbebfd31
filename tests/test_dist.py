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
