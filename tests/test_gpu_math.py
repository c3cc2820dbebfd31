"""Device-side building blocks against libm / the oracle, value by value (through cardiac_probe):
the branch-free exp and reciprocal that replace CUDA's exp() and division inside tanh and the
blended time constants, H_k, and the pointwise reactions N[z]
of the three models over their whole printed state ranges and beyond.
"""
import numpy as np
import pytest

import oracle as O
from paper_1309_1720_b200 import workloads as W

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def C():
    import torch
    assert torch.cuda.is_available()
    from paper_1309_1720_b200 import cardiac
    return cardiac


def probe(C, model, what, x, variant=0, nout=None):
    import torch
    cfg = W.make_config("probe", model, 8, W.LAP5, W.EULER, 0, variant=variant)
    xd = torch.from_numpy(np.ascontiguousarray(x, dtype=np.float64)).cuda()
    od = torch.empty_like(xd)
    n = x.shape[0]
    with C.Context.from_config(cfg) as ctx:
        C.cardiac_probe(ctx.ctx, what, xd, od, n)
        torch.cuda.synchronize()
    return od.cpu().numpy()


def test_exp_matches_libm_to_2ulp(C):
    rng = np.random.default_rng(5)
    x = np.concatenate([rng.uniform(-700, 700, 200000), rng.uniform(-2, 2, 200000),
                        rng.uniform(-1e-6, 1e-6, 1000), [0.0, 700.0, -700.0, 1.0, -1.0, 0.5 * np.log(2.0)]])
    got = probe(C, W.FHN, C.CARDIAC_PROBE_EXP, x)
    ref = np.exp(x)
    assert np.max(np.abs(got - ref) / ref) <= 2 * 2.3e-16
    # |x| limited to [700, 700.000123) beyond +-700 (high word clamped): finite, and the logistic built on it
    # is at its 0 / 1 limit there
    out = probe(C, W.FHN, C.CARDIAC_PROBE_EXP, np.array([1e4, -1e4, 5e300, -5e300]))
    assert np.all(np.isfinite(out)) and np.all(out[[0, 2]] >= np.exp(700.0)) and np.all(out[[0, 2]] < np.exp(700.001))
    assert np.all(out[[1, 3]] <= np.exp(-700.0)) and np.all(out[[1, 3]] > np.exp(-700.001))


def test_reciprocal_to_1ulp(C):
    rng = np.random.default_rng(6)
    x = np.concatenate([10.0 ** rng.uniform(-300, 300, 200000), rng.uniform(0.5, 2000.0, 200000)])
    got = probe(C, W.FHN, C.CARDIAC_PROBE_RCP, x)
    assert np.max(np.abs(got * x - 1.0)) <= 2.3e-16 * 1.5


def test_hk_matches_oracle(C):
    rng = np.random.default_rng(7)
    x = np.concatenate([rng.uniform(-0.03, 0.03, 20000), rng.uniform(-2, 2, 2000),
                        [-0.5 / 28.4, 0.0, 0.5 / 28.4]])
    got = probe(C, W.BOCF, C.CARDIAC_PROBE_HK, x)
    ref = np.array([O.hk(v, 28.4) for v in x])
    assert np.max(np.abs(got - ref)) <= 4e-16


@pytest.mark.parametrize("model,variant", [(W.FHN, 0), (W.KARMA, 0), (W.KARMA, 1), (W.BOCF, 0), (W.BOCF, 1)])
def test_reaction_matches_oracle_pointwise(C, model, variant):
    """Every branch of every H_k and both tails of every tanh: u sampled densely across the
    thresholds and well outside the printed ranges, gates in and slightly outside [0, 1]."""
    rng = np.random.default_rng(100 + model)
    nv = W.NUM_FIELDS[model]
    n = 60000
    lo, hi = {W.FHN: (-1.5, 1.5), W.KARMA: (-0.5, 4.5), W.BOCF: (-0.3, 2.0)}[model]
    z = np.empty((n, nv))
    z[:, 0] = rng.uniform(lo, hi, n)
    z[: n // 3, 0] = rng.uniform(-0.05, 0.45, n // 3) if model == W.BOCF else z[: n // 3, 0]
    for q in range(1, nv):
        z[:, q] = rng.uniform(-0.1, 1.2, n)
    z[-4:, 0] = [-30.0, 40.0, -8.0, 12.0]          # saturated tanh tails
    got = probe(C, model, C.CARDIAC_PROBE_REACTION, z, variant=variant)
    ref = np.array([O.reaction(model, zi, variant=variant) for zi in z])
    scale = np.maximum(1.0, np.abs(ref))
    assert np.max(np.abs(got - ref) / scale) <= 2e-13


def test_fp64_peak_and_issue_probe(C):
    """The measured FP64 peak (include/cardiac_diag.h) is within reach of the nominal 148 x 64 x 1.965 GHz, and an
    FP64 instruction does not share its issue slot: each integer instruction between two DFMAs costs about one
    more cycle (the model behind DESIGN.md "FP64 issue")."""
    cfg = W.make_config("probe", W.FHN, 8, W.LAP5, W.EULER, 0)
    with C.Context.from_config(cfg) as ctx:
        peak = C.cardiac_measure_fp64_peak(ctx.ctx, 2000, 3)
        r = [C.cardiac_measure_fp64_issue(ctx.ctx, m, 2000, 3) for m in (0, 2, 4)]
        with pytest.raises(C.CardiacError):
            C.cardiac_measure_fp64_issue(ctx.ctx, 3, 10, 1)
    nominal = 148 * 64 * 1.965e9
    assert 0.6 * nominal < peak <= 1.02 * nominal
    assert 0.8 * peak < r[0] <= 1.05 * peak
    assert r[0] > 1.4 * r[1] and r[1] > 1.3 * r[2]      # 2 : ~3.7 : ~6 cycles per DFMA
