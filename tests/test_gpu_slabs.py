"""One grid cut into row slabs (include/cardiac.h cardiac_get_rows / _set_rows;
paper_1309_1720_b200/dist.py): several contexts on ONE B200 stand for the ranks, stepped one after the
other, ghost rows moved device to device through the C ABI.  The own rows of the slabs must be the
undivided grid's result bit for bit — same kernels, same inputs, and the artificial edges of the
extended slabs only ever reach ghost rows."""
import numpy as np
import pytest

import oracle as O
from paper_1309_1720_b200 import dist as D
from paper_1309_1720_b200 import workloads as W

pytestmark = pytest.mark.gpu

STAGES = {W.EULER: 1, W.HEUN: 2, W.RK4: 4, W.RUSH_LARSEN: 1, W.IMPLICIT_EULER: 1}


@pytest.fixture(scope="module")
def C():
    import torch
    assert torch.cuda.is_available(), "gpu tests need a CUDA device"
    from paper_1309_1720_b200 import cardiac
    return cardiac


class _CtxStepper:
    def __init__(self, C, cfg, rows, Zext, plan):
        import torch
        self.torch = torch
        self.ctx = C.Context(cfg.model, cfg.nx, rows, cfg.dx, cfg.dt, cfg.scheme, cfg.batch, plan=plan)
        self.ctx.set_state(np.ascontiguousarray(Zext))
        self.shape = (cfg.batch, cfg.n_v, cfg.nx)

    def step(self, n):
        self.ctx.step(n)

    def get_rows(self, j0, n, dst=None):
        if dst is None:
            dst = self.torch.empty((self.shape[0], self.shape[1], n, self.shape[2]), dtype=self.torch.float64, device="cuda")
        return self.ctx.get_rows(j0, n, dst)

    def set_rows(self, j0, src):
        self.ctx.set_rows(j0, src)


@pytest.mark.parametrize("model,stencil,integ,plan,bc,world,every", [
    (W.FHN, W.LAP9X4, W.RK4, 0, 0, 2, 1),          # AUTO = FUSED
    (W.FHN, W.LAP9X4, W.RK4, 0, 1, 3, 1),          # periodic: every slab has two neighbours
    (W.BOCF, W.LAP9X4, W.RK4, 1, 0, 3, 1),         # STAGE
    (W.BOCF, W.LAP9X4, W.RK4, 4, 0, 2, 1),         # PAIR
    (W.KARMA, W.LAP5, W.HEUN, 0, 1, 2, 3),         # one exchange per 3 steps: 6 ghost rows
    (W.BOCF, W.BOX9, W.RUSH_LARSEN, 0, 0, 4, 2),
    (W.KARMA, W.BOX9, W.EULER, 2, 0, 2, 4),        # temporally blocked Euler, 4 steps per exchange
])
def test_slabs_equal_single_grid_bitwise(C, model, stencil, integ, plan, bc, world, every):
    cfg = W.make_config("slab", model, 70, stencil, integ, 0, batch=2, seed=6, ny=120, boundary=bc)
    Z = W.initial_state(cfg)
    nsteps = 12
    g = D.ghost_depth(2 if stencil == W.LAP9X4 else 1, STAGES[integ], every)
    slabs = [D.slab_of(cfg.ny, r, world, g, bool(bc)) for r in range(world)]
    steppers = [_CtxStepper(C, cfg, s.ext_rows, Z[:, :, s.global_rows(), :], plan) for s in slabs]
    left = nsteps
    while left > 0:
        n = min(every, left)
        for st in steppers:
            st.step(n)
        left -= n
        if left > 0:
            D.exchange_local(steppers, slabs)
    got = np.concatenate([st.ctx.get_rows(s.g_lo, s.own) for st, s in zip(steppers, slabs)], axis=2)
    for st in steppers:
        st.ctx.close()
    with C.Context.from_config(cfg, plan=plan) as ctx:
        ctx.set_state(Z)
        ctx.step(nsteps)
        whole = ctx.get_state()
    assert np.array_equal(got, whole)
    assert float(np.max(np.abs(got - O.step(model, Z, cfg.dx, cfg.dt, cfg.scheme, nsteps)))) <= 1e-12 * 10 * nsteps


def test_get_rows_writes_straight_into_another_contexts_memory(C):
    """include/cardiac.h: a DEVICE destination of cardiac_get_rows may be any address the GPU can store
    to — e.g. a peer's buffer mapped over NVLink, so that the pack kernel IS the transfer.  One GPU here:
    the destination is memory owned by ANOTHER context's caller-provided workspace region (as a peer's
    receive buffer would be), written by the sender's pack kernel on the sender's stream, consumed by
    the receiver's set_rows on ITS stream after an event — no host copy, no staging, no NCCL."""
    import torch
    cfg = W.make_config("peer", W.FHN, 70, W.LAP9X4, W.RK4, 0, batch=2, seed=9, ny=64)
    Z = W.initial_state(cfg)
    g = D.ghost_depth(2, 4)                                     # 8 ghost rows per cut
    slabs = [D.slab_of(cfg.ny, r, 2, g) for r in range(2)]
    streams = [torch.cuda.Stream(), torch.cuda.Stream()]
    ctxs, inbox = [], []
    for s, st in zip(slabs, streams):
        with torch.cuda.stream(st):
            c = C.Context(cfg.model, cfg.nx, s.ext_rows, cfg.dx, cfg.dt, cfg.scheme, cfg.batch)
            c.set_state(np.ascontiguousarray(Z[:, :, s.global_rows(), :]))
            # the receive buffer lives next to the receiver's workspace, in the receiver's allocation
            inbox.append(torch.empty((cfg.batch, cfg.n_v, g, cfg.nx), dtype=torch.float64, device="cuda"))
            ctxs.append(c)
    torch.cuda.synchronize()
    for step in range(6):
        done = []
        for r, (c, st) in enumerate(zip(ctxs, streams)):
            with torch.cuda.stream(st):
                c.step(1)
                # own rows next to the cut -> the OTHER context's inbox
                j0, n = slabs[r].send_to_upper() if r == 0 else slabs[r].send_to_lower()
                c.get_rows(j0, n, inbox[1 - r])
                ev = torch.cuda.Event(); ev.record(st); done.append(ev)
        for r, (c, st) in enumerate(zip(ctxs, streams)):
            with torch.cuda.stream(st):
                st.wait_event(done[1 - r])
                c.set_rows((slabs[r].recv_from_upper() if r == 0 else slabs[r].recv_from_lower())[0], inbox[r])
        torch.cuda.synchronize()
    got = np.concatenate([c.get_rows(s.g_lo, s.own) for c, s in zip(ctxs, slabs)], axis=2)
    for c in ctxs:
        c.close()
    with C.Context.from_config(cfg) as ctx:
        ctx.set_state(Z); ctx.step(6)
        whole = ctx.get_state()
    assert np.array_equal(got, whole)


def test_rows_roundtrip_and_errors(C):
    import torch
    cfg = W.make_config("rows", W.BOCF, 37, W.LAP5, W.RK4, 0, batch=3, seed=2, ny=29)
    Z = W.initial_state(cfg)
    with C.Context.from_config(cfg) as ctx:
        with pytest.raises(C.CardiacError) as ei:
            ctx.get_rows(0, 2)
        assert ei.value.code == C.CARDIAC_ERR_NOSTATE
        ctx.set_state(Z)
        assert np.array_equal(ctx.get_rows(5, 7), Z[:, :, 5:12, :])            # host destination
        d = torch.empty((3, 4, 4, 37), dtype=torch.float64, device="cuda")
        ctx.get_rows(25, 4, d)                                                 # device destination, last rows
        torch.cuda.synchronize()
        assert np.array_equal(d.cpu().numpy(), Z[:, :, 25:29, :])
        new = np.ascontiguousarray(np.arange(3 * 4 * 2 * 37, dtype=np.float64).reshape(3, 4, 2, 37))
        ctx.set_rows(10, new)
        ctx.set_rows(0, torch.from_numpy(new).cuda() + 0.5)
        Z2 = Z.copy(); Z2[:, :, 10:12, :] = new; Z2[:, :, 0:2, :] = new + 0.5
        assert np.array_equal(ctx.get_state(), Z2)
        assert ctx.get_rows(3, 0).shape == (3, 4, 0, 37)
        for j0, n in [(-1, 2), (28, 2), (0, 30), (5, -1)]:
            with pytest.raises(C.CardiacError) as ei:
                ctx.get_rows(j0, n, np.empty((3, 4, max(n, 0), 37)))
            assert ei.value.code == C.CARDIAC_ERR_INVALID
    # 3-D: a row index runs over (plane, row); a slab of planes is a row range
    cfg3 = W.make_config("rows3", W.FHN, 12, W.LAP5, W.EULER, 0, seed=3, ny=10, nz=9)
    Z3 = W.initial_state(cfg3)
    with C.Context.from_config(cfg3) as ctx:
        ctx.set_state(Z3)
        assert np.array_equal(ctx.get_rows(2 * 10, 3 * 10).reshape(1, 2, 3, 10, 12), Z3[:, :, 2:5])


def test_3d_slabs_of_planes_equal_single_grid_bitwise(C):
    """3-D: the cut runs between planes; a ghost plane is ny rows of the flattened index."""
    import dataclasses
    import torch
    cfg = W.make_config("slab3", W.KARMA, 20, W.LAP9X4, W.RK4, 0, seed=8, ny=14, nz=40)
    cfg = dataclasses.replace(cfg, dt=W.default_dt_3d(W.KARMA))
    Z = W.initial_state(cfg)                                   # [1][2][nz][ny][nx]
    world, nsteps = 2, 5
    g = D.ghost_depth(2, 4)
    slabs = [D.slab_of(cfg.nz, r, world, g) for r in range(world)]

    class PlaneStepper:
        def __init__(self, s):
            self.ctx = C.Context(cfg.model, cfg.nx, cfg.ny, cfg.dx, cfg.dt, cfg.scheme, 1, nz=s.ext_rows)
            self.ctx.set_state(np.ascontiguousarray(Z[:, :, s.global_rows()]))
        def step(self, n):
            self.ctx.step(n)
        def get_rows(self, p0, n, dst=None):
            dst = torch.empty((1, cfg.n_v, n * cfg.ny, cfg.nx), dtype=torch.float64, device="cuda")
            return self.ctx.get_rows(p0 * cfg.ny, n * cfg.ny, dst)
        def set_rows(self, p0, src):
            self.ctx.set_rows(p0 * cfg.ny, src)

    steppers = [PlaneStepper(s) for s in slabs]
    for k in range(nsteps):
        for st in steppers:
            st.step(1)
        if k + 1 < nsteps:
            D.exchange_local(steppers, slabs)
    got = np.concatenate([st.ctx.get_state()[:, :, s.g_lo:s.g_lo + s.own] for st, s in zip(steppers, slabs)], axis=2)
    for st in steppers:
        st.ctx.close()
    with C.Context.from_config(cfg) as ctx:
        ctx.set_state(Z)
        ctx.step(nsteps)
        whole = ctx.get_state()
    assert np.array_equal(got, whole)
