"""Host logic of the seeded input generators (no GPU, no oracle arithmetic)."""
import numpy as np
import pytest

from paper_1309_1720_b200 import workloads as W


def test_rng_is_counter_based_and_reproducible():
    a = W.uniform01(3, 1000)
    assert np.array_equal(a, W.uniform01(3, 1000))
    assert np.array_equal(a[:100], W.uniform01(3, 100))         # independent of how many are drawn
    assert not np.array_equal(a, W.uniform01(4, 1000))
    assert not np.array_equal(a, W.uniform01(3, 1000, stream=1))
    assert a.min() >= 0.0 and a.max() < 1.0 and abs(a.mean() - 0.5) < 0.05
    g = W.gaussian(9, 200_000)
    assert abs(g.mean()) < 0.01 and abs(g.std() - 1.0) < 0.01


def test_baseline_configs_follow_baseline_json():
    c = [W.baseline_config(i) for i in range(1, 6)]
    assert [(x.model, x.nx, x.ny, x.stencil, x.integrator, x.nsteps, x.batch) for x in c] == [
        (W.FHN, 64, 64, W.LAP5, W.EULER, 200, 1),
        (W.FHN, 512, 512, W.LAP9X4, W.RK4, 10_000, 1),
        (W.KARMA, 1024, 1024, W.LAP5, W.RK4, 5_000, 1),
        (W.BOCF, 2048, 2048, W.LAP9X4, W.RK4, 2_000, 1),
        (W.FHN, 512, 512, W.LAP9X4, W.RK4, 1_000, 17)]
    # dt = 0.5 * dx^2 / (4 D_max)  (BASELINE.json:configs[0])
    assert c[0].dt == pytest.approx(0.5 * 0.04 ** 2 / (4 * 1.5), rel=1e-15)
    assert c[2].dt == pytest.approx(0.0780045454545, rel=1e-9)
    assert c[3].dt == pytest.approx(0.0960717335611, rel=1e-9)
    assert c[1].scheme == 1 | (2 << 8)
    with pytest.raises(ValueError):
        W.baseline_config(6)


def test_initial_states():
    c1 = W.baseline_config(1)
    z = W.initial_state(c1)
    assert z.shape == (1, 2, 64, 64) and z.dtype == np.float64
    assert np.all(np.abs(z[0, 0, :, :5] - 1.0) <= 1e-3) and np.all(np.abs(z[0, 0, :, 5:] - W.REST[W.FHN][0]) <= 1e-3)
    assert np.all(np.abs(z[0, 1] - W.REST[W.FHN][1]) <= 1e-3) and z[0, 1].std() > 1e-4
    assert np.array_equal(z, W.initial_state(c1))

    c2 = W.scaled(W.baseline_config(2), 32)
    z = W.initial_state(c2)[0]
    assert np.allclose(z[0, :16, :16], 1.0, atol=1e-5) and np.allclose(z[0, 16:, :], W.REST[W.FHN][0], atol=1e-5)
    assert np.allclose(z[1, 16:, :], 0.0219, atol=1e-3) and np.allclose(z[1, :16, :], W.REST[W.FHN][1], atol=1e-5)

    c3 = W.scaled(W.baseline_config(3), 48, ny=40)
    z = W.initial_state(c3)[0]
    assert z.shape == (2, 40, 48)
    assert 0.0 <= z[0].min() and z[0].max() <= 3.5 and 0.0 <= z[1].min() and z[1].max() <= 1.0
    assert np.abs(np.diff(z[0], axis=1)).max() < 1.5      # smoothed: no raw block edges

    c4 = W.scaled(W.baseline_config(4), 32)
    z = W.initial_state(c4)
    assert np.all(z[0, 0, :, :8] == 1.0) and np.all(z[0, 0, :, 8:] == 0.0)
    for f in (1, 2, 3):
        assert np.all(z[0, f] == W.REST[W.BOCF][f])
    s = W.stimulus_cfg4(z)
    assert np.all(s[0, 0, :16, :] == 1.0) and np.array_equal(s[0, 1:], z[0, 1:]) and np.array_equal(s[0, 0, 16:], z[0, 0, 16:])

    c5 = W.scaled(W.baseline_config(5), 24)
    z = W.initial_state(c5)
    assert z.shape == (17, 2, 24, 24)
    d = (z[1:] - z[0]) / 1e-7
    assert np.allclose(np.sqrt(np.sum(d ** 2, axis=(1, 2, 3))), 1.0, atol=1e-6)
    assert abs(np.sum(d[0] * d[1])) < 0.2                 # different directions
    # full size: the base is BASELINE.json:configs[4]'s "config-2 state after 5000 RK4 steps", never a stand-in
    c5f = W.baseline_config(5)
    with pytest.raises(ValueError):
        W.initial_state(c5f)
    one, z2, n = W.base_recipe_cfg5(c5f)
    assert n == 5000 and (one.batch, one.nx, one.ny, one.integrator, one.stencil) == (1, 512, 512, W.RK4, W.LAP9X4)
    assert np.array_equal(z2, W.initial_state(W.baseline_config(2)))
    zf = W.initial_state(c5f, base=z2[0])
    assert zf.shape == (17, 2, 512, 512) and np.array_equal(zf[0], z2[0])


def test_sweep_and_3d_inputs():
    """Size sweep S and the 3-D inputs: shapes, determinism, value ranges."""
    assert W.sweep_sizes()[0] == 64 and 362 in W.sweep_sizes() and W.sweep_sizes()[-1] == 8192
    c = W.sweep_config(W.KARMA, 362)
    assert (c.stencil, c.integrator, c.nsteps) == (W.LAP5, W.RK4, 200) and W.sweep_config(W.BOCF, 8192).nsteps == 32
    z = W.sweep_state(c)
    assert z.shape == (1, 2, 362, 362) and np.array_equal(z, W.sweep_state(c))
    assert np.array_equal(z[0, :, :106, :106], z[0, :, 256:362, 256:362])     # the 256^2 base, repeated
    lo, hi = W.U_RANGE[W.KARMA]
    assert lo <= z[0, 0].min() and z[0, 0].max() <= hi
    c3 = W.make_config("v", W.BOCF, 20, W.LAP9X4, W.RK4, 0, batch=2, seed=4, ny=12, nz=7)
    assert c3.cells == 2 * 20 * 12 * 7
    z3 = W.initial_state(c3)
    assert z3.shape == (2, 4, 7, 12, 20) and np.array_equal(z3, W.initial_state(c3))
    assert not np.array_equal(z3[0, 0, 0], z3[0, 0, 3])                        # planes differ
    assert 0 < np.max(np.abs(z3[1] - z3[0])) < 1e-2                             # perturbed batch member
    assert W.default_dt_3d(W.FHN) == pytest.approx(0.5 * 0.04 ** 2 / (6 * 1.5), rel=1e-15)
