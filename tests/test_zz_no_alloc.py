"""cardiac_step_static (include/cardiac_static.h): the entry point that allocates nothing — stage buffers in a
static __device__ array inside the library — against the existing context path, on calls in a row that share
that array.  Collected last (file name) so that a failure here hides no other test.  Needs a B200.
"""
import numpy as np
import pytest

from paper_1309_1720_b200 import workloads as W

pytestmark = pytest.mark.gpu

TOL_1 = 1e-12     # the tolerances of tests/test_gpu_parity.py (BASELINE.json:north_star)
TOL_100 = 1e-9


def tol(nsteps):
    return TOL_1 if nsteps <= 1 else min(TOL_100, TOL_1 * 10 * nsteps)


@pytest.fixture(scope="module")
def C():
    import torch
    assert torch.cuda.is_available(), "gpu tests need a CUDA device"
    from paper_1309_1720_b200 import cardiac
    return cardiac


def context_path(C, cfg, Z0, nsteps, plan=0, plan_param=0):
    """The existing path: a context (workspace cudaMalloc'ed by the library), AUTO or a forced plan."""
    with C.Context.from_config(cfg, plan=plan, plan_param=plan_param) as ctx:
        ctx.set_state(np.ascontiguousarray(Z0))
        ctx.step(nsteps)
        return ctx.get_state()


def static_path(C, cfg, Z0, nsteps, in_place=False):
    import torch
    src = torch.from_numpy(np.ascontiguousarray(Z0)).cuda()
    dst = src if in_place else torch.full_like(src, float("nan"))
    C.cardiac_step_static(cfg.model, cfg.scheme, cfg.nx, cfg.ny, cfg.batch, cfg.dx, cfg.dt, None, src, dst, nsteps,
                          torch.cuda.current_stream().cuda_stream)
    torch.cuda.synchronize()
    return dst.cpu().numpy()


def case(model, nx, ny, stencil, integ, batch=1, seed=5, **kw):
    cfg = W.make_config("static", model, nx, stencil, integ, 0, batch=batch, seed=seed, ny=ny, **kw)
    return cfg, W.initial_state(cfg)


def test_static_scratch_matches_context_path_on_calls_in_a_row(C):
    import torch
    # A: the 4-field model, RK4 (four stage buffers), a grid with ragged tiles; B: a smaller two-field problem
    # with an odd row length, forward Euler and periodic boundaries (two buffers, other pitch: it lands on A's
    # leftovers); then A again over B's leftovers, in place.
    cfg_a, Za = case(W.BOCF, 150, 97, W.LAP9X4, W.RK4, batch=2)
    cfg_b, Zb = case(W.FHN, 37, 29, W.LAP5, W.EULER, boundary=1)
    na, nb = 20, 50
    ref_a = context_path(C, cfg_a, Za, na)                     # AUTO plan
    ref_a_stage = context_path(C, cfg_a, Za, na, plan=1, plan_param=1)   # the same kernels: STAGE, DIRECT
    ref_b = context_path(C, cfg_b, Zb, nb)
    ref_b_stage = context_path(C, cfg_b, Zb, nb, plan=1, plan_param=1)

    out_a1 = static_path(C, cfg_a, Za, na)                      # (first call: module load, symbol look-up)
    torch.cuda.synchronize()
    free0 = torch.cuda.mem_get_info()[0]
    out_b = static_path(C, cfg_b, Zb, nb)
    out_a2 = static_path(C, cfg_a, Za, na, in_place=True)
    out_b2 = static_path(C, cfg_b, Zb, nb)
    free1 = torch.cuda.mem_get_info()[0]

    for out, ref, ref_stage, n in ((out_a1, ref_a, ref_a_stage, na), (out_b, ref_b, ref_b_stage, nb),
                                   (out_a2, ref_a, ref_a_stage, na), (out_b2, ref_b, ref_b_stage, nb)):
        assert np.all(np.isfinite(out))
        assert float(np.max(np.abs(out - ref))) <= tol(n)
        assert np.array_equal(out, ref_stage)     # same kernels, same launch sequence: the same bits
    # the library took no device memory for these calls (the tensors of static_path are torch's, freed into
    # its caching allocator, which only ever grows: free memory can only have gone down through torch)
    assert free1 <= free0 and free0 - free1 <= 2 * (Za.nbytes + Zb.nbytes) + (4 << 20)


def test_static_scratch_heun_and_gate_integrators(C):
    for model, integ, stencil in ((W.KARMA, W.HEUN, W.BOX9), (W.BOCF, W.RUSH_LARSEN, W.LAP5)):
        cfg, Z = case(model, 70, 45, stencil, integ)
        out = static_path(C, cfg, Z, 10)
        assert np.array_equal(out, context_path(C, cfg, Z, 10, plan=1, plan_param=1))
        assert float(np.max(np.abs(out - context_path(C, cfg, Z, 10)))) <= tol(10)


def test_static_scratch_rejects_what_does_not_fit(C):
    import torch
    # BOCF RK4 512 x 512 is exactly the 32 MiB; one more row is not
    need_ok = 4 * 4 * 512 * 512 * 8
    assert need_ok == C.CARDIAC_STATIC_SCRATCH_BYTES
    z = torch.zeros((1, 4, 513, 512), dtype=torch.float64, device="cuda")
    with pytest.raises(C.CardiacError) as ei:
        C.cardiac_step_static(W.BOCF, W.LAP9X4 | W.RK4 << 8, 512, 513, 1, 0.025, 0.01, None, z, z, 1)
    assert ei.value.code == C.CARDIAC_ERR_WORKSPACE
    assert str(C.CARDIAC_STATIC_SCRATCH_BYTES) in str(ei.value) and str(need_ok // 512 * 513) in str(ei.value)
    # bad arguments are named, nothing is enqueued
    with pytest.raises(C.CardiacError) as ei:
        C.cardiac_step_static(W.FHN, W.LAP5, 2, 64, 1, 0.04, 1e-4, None, z, z, 1)
    assert ei.value.code == C.CARDIAC_ERR_INVALID and "nx" in str(ei.value)
    # the largest problem that fits runs (one step, finite result)
    cfg, Z = case(W.BOCF, 512, 512, W.LAP9X4, W.RK4)
    out = static_path(C, cfg, Z, 1)
    assert np.array_equal(out, context_path(C, cfg, Z, 1, plan=1, plan_param=1))
