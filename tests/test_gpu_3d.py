"""3-D grids through the C ABI (cardiac_create3d) against the 3-D
oracle, element by element, at the tolerances of the 2-D path.  Needs a B200.
"""
import dataclasses

import numpy as np
import pytest

import oracle as O
from paper_1309_1720_b200 import workloads as W

pytestmark = pytest.mark.gpu

TOL_1, TOL_100 = 1e-12, 1e-9


def tol(nsteps):
    """1e-12 at one step, 1e-9 at 100 (north_star), linear in between: TOL_1 x 10 x nsteps."""
    return TOL_1 if nsteps <= 1 else min(TOL_100, TOL_1 * 10 * nsteps)
FHN, KARMA, BOCF = W.FHN, W.KARMA, W.BOCF
LAP5, LAP9X4, BOX9 = W.LAP5, W.LAP9X4, W.BOX9
EULER, HEUN, RK4, RL, IE = W.EULER, W.HEUN, W.RK4, W.RUSH_LARSEN, W.IMPLICIT_EULER


@pytest.fixture(scope="module")
def C():
    import torch
    assert torch.cuda.is_available(), "gpu tests need a CUDA device"
    from paper_1309_1720_b200 import cardiac
    return cardiac


def make(model, nx, ny, nz, stencil, integ, batch=1, seed=13, **kw):
    cfg = W.make_config("case3d", model, nx, stencil, integ, 0, batch=batch, seed=seed, ny=ny, nz=nz, **kw)
    cfg = dataclasses.replace(cfg, dt=W.default_dt_3d(model))
    return cfg, W.initial_state(cfg)


DIRECT, RING = 1, 2     # plan STAGE: every thread loads its operands / z-marching persistent CTAs fed by a TMA ring


def gpu_run(C, cfg, Z, nsteps, chunks=None, impl=0):
    with C.Context.from_config(cfg, plan=1 if impl else 0, plan_param=impl) as ctx:
        assert ctx.plan == 1                                   # 3-D runs the stage-synchronous plan
        ctx.set_state(np.ascontiguousarray(Z))
        for n in (chunks or [nsteps]):
            ctx.step(n)
        out = ctx.get_state()
    return out


def maxabs(a, b):
    return float(np.max(np.abs(a - b)))


CASES = [(m, s, i) for m in (FHN, KARMA, BOCF) for s in (LAP5, LAP9X4) for i in (EULER, HEUN, RK4)]
CASES += [(BOCF, s, i) for s in (LAP5, LAP9X4) for i in (RL, IE)]


@pytest.mark.parametrize("model,stencil,integ", CASES)
def test_parity_3d_one_and_fifty_steps(C, model, stencil, integ):
    # 141 x 27 x 7: interior blocks (x, y and z) as well as rim blocks on every face, odd width
    cfg, Z = make(model, 141, 27, 7, stencil, integ)
    got1 = gpu_run(C, cfg, Z, 1, impl=DIRECT)
    ref1 = O.step3d(model, Z, cfg.dx, cfg.dt, cfg.scheme, 1, omp=True)
    assert maxabs(got1, ref1) <= TOL_1
    got = gpu_run(C, cfg, Z, 50, impl=DIRECT)
    ref = O.step3d(model, ref1, cfg.dx, cfg.dt, cfg.scheme, 49, omp=True)
    assert np.all(np.isfinite(got))
    assert maxabs(got, ref) <= tol(50)
    assert maxabs(got, Z) > 1e-6
    if integ in (EULER, HEUN, RK4):     # the TMA ring marching along z: the same arithmetic per cell, the same bits
        assert np.array_equal(gpu_run(C, cfg, Z, 50, impl=RING), got)


@pytest.mark.parametrize("model,stencil,nx,ny,nz,bc", [(FHN, LAP9X4, 200, 70, 75, 0), (KARMA, LAP5, 130, 19, 40, 1),
                                                       (BOCF, LAP9X4, 67, 9, 33, 0), (FHN, LAP5, 64, 8, 32, 1),
                                                       (FHN, LAP9X4, 65, 17, 5, 1)])
def test_parity_3d_ring_chunks_and_tiles(C, model, stencil, nx, ny, nz, bc):
    """The z-marching ring on grids of several 64 x 8 tiles and more than one chunk of 32 planes (75 = 32 + 32 + 11),
    exactly one tile and one chunk, fewer planes than ring slots, ragged tiles, batch of 2: against the oracle and
    bitwise against the direct kernels."""
    cfg, Z = make(model, nx, ny, nz, stencil, RK4, boundary=bc, batch=2)
    got = gpu_run(C, cfg, Z, 6, impl=RING)
    assert np.array_equal(got, gpu_run(C, cfg, Z, 6, impl=DIRECT))
    assert maxabs(got, O.step3d(model, Z, cfg.dx, cfg.dt, cfg.scheme, 6, omp=True)) <= tol(6)


@pytest.mark.parametrize("model,stencil,nx,ny,nz,bc", [(FHN, LAP5, 3, 3, 3, 0), (KARMA, LAP9X4, 5, 5, 5, 0),
                                                       (BOCF, LAP9X4, 37, 6, 5, 1), (FHN, LAP9X4, 140, 30, 9, 1),
                                                       (KARMA, LAP5, 8, 70, 3, 0)])
def test_parity_3d_edges_and_periodic(C, model, stencil, nx, ny, nz, bc):
    """Minimum sizes 2r+1 in every direction (every arm reflects), thin slabs, periodic wrap in z."""
    cfg, Z = make(model, nx, ny, nz, stencil, RK4, boundary=bc)
    got = gpu_run(C, cfg, Z, 20, impl=DIRECT)
    ref = O.step3d(model, Z, cfg.dx, cfg.dt, cfg.scheme, 20)
    assert maxabs(got, ref) <= tol(20)
    assert np.array_equal(gpu_run(C, cfg, Z, 20, impl=RING), got)


def test_3d_batch_jvp_and_composition(C):
    cfg, Z = make(FHN, 70, 20, 6, LAP9X4, RK4, batch=4, seed=2)
    got = gpu_run(C, cfg, Z, 12)
    ref = O.step3d(FHN, Z, cfg.dx, cfg.dt, cfg.scheme, 12)
    assert maxabs(got, ref) <= tol(12)
    perm = [2, 0, 3, 1]
    assert np.array_equal(gpu_run(C, cfg, Z[perm], 12), got[perm])          # whatever the slot
    assert np.array_equal(gpu_run(C, cfg, Z, 12, chunks=[1, 5, 6]), got)     # step(a); step(b) == step(a+b)
    with C.Context.from_config(cfg) as ctx:
        ctx.set_state(Z); ctx.step(12)
        J = ctx.get_jvp(1e-7)
    assert J.shape == (3, 2, 6, 20, 70)
    assert np.array_equal(J, (got[1:] - got[0]) / 1e-7)


def test_3d_z_independent_state_matches_2d_run(C):
    """Identical planes: the z arm of the stencil cancels (to rounding of the 13-point weights) and every
    plane follows the 2-D path."""
    cfg, _ = make(KARMA, 96, 40, 6, LAP9X4, RK4)
    cfg2 = dataclasses.replace(cfg, nz=1)
    plane = W.state_blocks(cfg2)                                   # [1][n_v][ny][nx]
    Z = np.repeat(plane[:, :, None], 6, axis=2)
    got3 = gpu_run(C, cfg, Z, 30)
    with C.Context.from_config(cfg2, plan=1) as ctx:
        ctx.set_state(plane); ctx.step(30)
        got2 = ctx.get_state()
    for k in range(6):
        assert maxabs(got3[:, :, k], got2) <= 1e-12


def test_3d_argument_checks(C):
    ok = dict(model=FHN, nx=16, ny=16, nz=8, dx=0.04, dt=1e-4, scheme=W.LAP9X4 | (W.RK4 << 8), batch=1)
    C.cardiac_destroy(C.cardiac_create3d(**ok))
    for bad in (dict(nz=4), dict(nz=0), dict(scheme=W.BOX9 | (W.RK4 << 8)), dict(batch=9000), dict(nz=-3)):
        with pytest.raises(C.CardiacError):
            C.cardiac_create3d(**{**ok, **bad})
    cfg, _ = make(FHN, 16, 16, 8, LAP5, RK4)
    with C.Context.from_config(cfg) as ctx:
        for plan in (2, 3, (1, 3)):
            with pytest.raises(C.CardiacError):
                C.cardiac_set_plan(ctx.ctx, *(plan if isinstance(plan, tuple) else (plan, 0)))
