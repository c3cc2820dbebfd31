"""Pins of the oracle's pointwise reactions N[z] and H_k (no GPU).

Expected values: numbers printed in the paper (tests/golden/paper_constants.json), closed forms
worked out by hand below, special cases in which every smoothed step is saturated (the models
reduce to their original sharp-Heaviside textbook form), fixed points, and printed field ranges.
Cites: PAPER.md:48-96; Q7-Q11.
"""
import json
import os

import numpy as np
import pytest

import oracle as O
from paper_1309_1720_b200 import workloads as W

FHN, KARMA, BOCF = 0, 1, 2
GOLD = json.load(open(os.path.join(os.path.dirname(__file__), "golden", "paper_constants.json")))


def smoothstep(x, k=28.4):
    """The standard cubic smoothstep of t = kx + 1/2 (Q11) — NOT the paper's branch form."""
    t = min(1.0, max(0.0, k * x + 0.5))
    return t * t * (3.0 - 2.0 * t)


# ----------------------------------------------------------------------------- printed constants
def test_defaults_match_printed_constants():
    p = O.default_params(FHN)
    g = GOLD["fhn"]
    assert (p[1], p[2], p[3], p[4]) == (g["delta"], g["epsilon"], g["a1"], g["a0"]) and p[0] == 1.0
    p = O.default_params(KARMA)
    g = GOLD["karma"]
    assert (p[6], p[7], p[0]) == (g["Re"], g["M"], g["gamma"]) and p[8] == GOLD["hk"]["k"]
    p = O.default_params(BOCF)
    assert p[0] == pytest.approx(GOLD["bocf"]["D_cm2_per_s"] * 1e-3, rel=1e-15)  # cm^2/s -> cm^2/ms
    assert p[1] == GOLD["hk"]["k"] and p[3] == GOLD["u_range"]["bocf"][1]
    assert W.DX == {FHN: GOLD["fhn"]["dx"], KARMA: GOLD["karma"]["dx"], BOCF: GOLD["bocf"]["dx"]}
    for m, name in ((FHN, "fhn"), (KARMA, "karma"), (BOCF, "bocf")):
        assert list(W.U_RANGE[m]) == GOLD["u_range"][name]
    assert [O.num_fields(m) for m in (0, 1, 2)] == [2, 2, 4]
    assert O.num_fields(7) == -1


def test_kernel_count_arithmetic():
    """(n_d + 2) n_s = 12 for Karma RK4 fixes n_d(Karma) = 1, n_s(RK4) = 4."""
    assert (W.NUM_DIFFUSING[KARMA] + 2) * W.STAGES[W.RK4] == GOLD["kernel_calls"]["karma_rk4"]
    assert (W.NUM_DIFFUSING[FHN] + 2) * W.STAGES[W.RK4] == 16


# ----------------------------------------------------------------------------- H_k
def test_hk_breakpoints_and_identities():
    k = GOLD["hk"]["k"]
    for kx, val in zip(GOLD["hk"]["breakpoints_kx"], GOLD["hk"]["values"]):
        assert O.hk(kx / k, k) == pytest.approx(val, abs=1e-15)
    assert O.hk(-1.0, k) == 0.0 and O.hk(1.0, k) == 1.0
    assert 1.0 / k == pytest.approx(GOLD["hk"]["width"], abs=5e-4)  # transition width w = 1/k ~ 0.035
    xs = np.linspace(-0.03, 0.03, 241)
    h = np.array([O.hk(x, k) for x in xs])
    assert np.all(np.diff(h) >= 0)                                   # monotone
    assert np.max(np.abs(h + h[::-1] - 1.0)) < 1e-15                 # H(x) + H(-x) = 1
    assert np.max(np.abs(h - [smoothstep(x, k) for x in xs])) < 1e-15  # = t^2 (3 - 2t)  (Q11)
    # C^1 at the breakpoints: one-sided slopes vanish there, 1.5 k at the centre
    e = 1e-7
    assert abs((O.hk(0.5 / k, k) - O.hk(0.5 / k - e, k)) / e) < 1e-3
    assert abs((O.hk(-0.5 / k + e, k) - O.hk(-0.5 / k, k)) / e) < 1e-3
    assert (O.hk(e, k) - O.hk(-e, k)) / (2 * e) == pytest.approx(1.5 * k, rel=1e-6)


# ----------------------------------------------------------------------------- FHN
def test_fhn_hand_values():
    # N_u = u - v - u^3, N_v = eps (u - a1 v - a0)
    f = O.reaction(FHN, [0.5, 0.1])
    assert f[0] == pytest.approx(0.5 - 0.1 - 0.125, abs=1e-16)
    assert f[1] == pytest.approx(0.05 * (0.5 - 0.15 + 0.1), abs=1e-17)
    f = O.reaction(FHN, [-2.0, 1.0])
    assert f[0] == pytest.approx(-2.0 - 1.0 + 8.0, abs=1e-15)
    assert f[1] == pytest.approx(0.05 * (-2.0 - 1.5 + 0.1), abs=1e-16)


def test_fhn_fixed_points_from_the_cubic():
    """u - (u - a0)/a1 - u^3 = 0: roots via numpy.roots."""
    a1, a0 = 1.5, -0.1
    roots = np.sort(np.roots([-1.0, 0.0, 1.0 - 1.0 / a1, a0 / a1]).real)
    assert roots == pytest.approx([-0.65914658116074, 0.24309975855228, 0.41604682260846], abs=1e-12)
    for u in roots:
        assert np.max(np.abs(O.reaction(FHN, [u, (u - a0) / a1]))) < 1e-15
    assert W.REST[FHN][0] == pytest.approx(roots[0], abs=1e-14)
    assert W.REST[FHN][1] == pytest.approx((roots[0] - a0) / a1, abs=1e-14)


# ----------------------------------------------------------------------------- Karma
def test_karma_hand_values():
    cR = 1.0 / (1.0 - np.exp(-1.0))
    # u = 3 = u_h: tanh(0) = 0; v = 0 -> (u^2/2 * u_star - u)/tau_u; u > u_v + 1/(2k): f_v = (cR - v)/tau_v
    f = O.reaction(KARMA, [3.0, 0.0])
    assert f[0] == pytest.approx((4.5 * 1.5415 - 3.0) / 2.5, abs=1e-15)
    assert f[1] == pytest.approx(cR / 250.0, abs=1e-17)
    # v = 1: v^M = 1
    f = O.reaction(KARMA, [3.0, 1.0])
    assert f[0] == pytest.approx((4.5 * 0.5415 - 3.0) / 2.5, abs=1e-15)
    assert f[1] == pytest.approx((cR - 1.0) / 250.0, abs=1e-17)
    # below threshold: f_v = -v/tau_v; tanh(-2.5)
    f = O.reaction(KARMA, [0.5, 0.8])
    assert f[1] == pytest.approx(-0.8 / 250.0, abs=1e-18)
    assert f[0] == pytest.approx((0.125 * (1.0 - np.tanh(-2.5)) * (1.5415 - 0.8 ** 6) - 0.5) / 2.5, abs=1e-15)
    # v^M with M = 6 and a NEGATIVE v is even
    assert O.reaction(KARMA, [2.0, -0.5])[0] == pytest.approx(O.reaction(KARMA, [2.0, 0.5])[0], abs=1e-16)
    # at u = u_v the two steps are both 1/2: f_v = (cR/2 - v)/tau_v
    assert O.reaction(KARMA, [1.0, 0.3])[1] == pytest.approx((0.5 * cR - 0.3) / 250.0, abs=1e-17)
    assert np.all(O.reaction(KARMA, [0.0, 0.0]) == 0.0)  # rest state exactly (0, 0)


def _single_cell(model, z0, dt, nsteps, record=0):
    """Scalar RK4 built on oracle.reaction only (no grid code)."""
    z = np.array(z0, dtype=float)
    trace = np.empty((nsteps + 1, z.size))
    trace[0] = z
    f = lambda y: O.reaction(model, y)
    for n in range(nsteps):
        k1 = f(z); k2 = f(z + dt / 2 * k1); k3 = f(z + dt / 2 * k2); k4 = f(z + dt * k3)
        z = z + dt / 6 * (k1 + 2 * k2 + 2 * k3 + k4)
        trace[n + 1] = z
    return trace


def test_karma_single_cell_ranges():
    """Excitable with threshold between u0 = 0.5 and 0.9; voltage stays in the printed range (0, 3.5)
    within ~10 %, gate in (0,1) within a few %."""
    lo, hi = GOLD["u_range"]["karma"]
    sub = _single_cell(KARMA, [0.5, 0.0], 0.1, 600)
    assert sub[-1, 0] < 0.05 and sub[:, 0].max() <= 0.5 + 1e-12
    ap = _single_cell(KARMA, [0.9, 0.0], 0.1, 8000)
    assert 0.9 * hi < ap[:, 0].max() < 1.12 * hi
    assert ap[:, 0].min() > lo - 1e-9
    assert 0.9 < ap[:, 1].max() < 1.1 and ap[:, 1].min() > -1e-12
    assert ap[-1, 0] < 0.05  # repolarised


# ----------------------------------------------------------------------------- BOCF
P = dict(u_o=0.0, u_u=1.55, th_v=0.3, th_w=0.13, th_vm=0.006, th_o=0.006, tv1m=60.0, tv2m=1150.0,
         tvp=1.4506, tw1m=60.0, tw2m=15.0, kwm=65.0, uwm=0.03, twp=200.0, tfi=0.11, to1=400.0,
         to2=6.0, tso1=30.0181, tso2=0.9957, kso=2.0458, uso=0.65, ts1=2.7342, ts2=16.0, ks=2.0994,
         us=0.9087, tsi=1.8875, twinf=0.07, winfs=0.94)


def _bocf_sharp(u, v, w, s):
    """The minimal model in its ORIGINAL Heaviside form (Ref. [3] of the paper), valid wherever
    every |k (u - theta)| > 1/2 so that all H_k are saturated."""
    H = lambda x: 1.0 if x > 0 else 0.0
    p = P
    tvm = (1 - H(u - p["th_vm"])) * p["tv1m"] + H(u - p["th_vm"]) * p["tv2m"]
    twm = p["tw1m"] + (p["tw2m"] - p["tw1m"]) * (1 + np.tanh(p["kwm"] * (u - p["uwm"]))) / 2
    tso = p["tso1"] + (p["tso2"] - p["tso1"]) * (1 + np.tanh(p["kso"] * (u - p["uso"]))) / 2
    ts = (1 - H(u - p["th_w"])) * p["ts1"] + H(u - p["th_w"]) * p["ts2"]
    to = (1 - H(u - p["th_o"])) * p["to1"] + H(u - p["th_o"]) * p["to2"]
    vinf = 1.0 if u < p["th_vm"] else 0.0
    winf = (1 - H(u - p["th_o"])) * (1 - u / p["twinf"]) + H(u - p["th_o"]) * p["winfs"]
    Jfi = -v * H(u - p["th_v"]) * (u - p["th_v"]) * (p["u_u"] - u) / p["tfi"]
    Jso = (u - p["u_o"]) * (1 - H(u - p["th_w"])) / to + H(u - p["th_w"]) / tso
    Jsi = -H(u - p["th_w"]) * w * s / p["tsi"]
    du = -(Jfi + Jso + Jsi)
    dv = (1 - H(u - p["th_v"])) * (vinf - v) / tvm - H(u - p["th_v"]) * v / p["tvp"]
    dw = (1 - H(u - p["th_w"])) * (winf - w) / twm - H(u - p["th_w"]) * w / p["twp"]
    ds = ((1 + np.tanh(p["ks"] * (u - p["us"]))) / 2 - s) / ts
    return np.array([du, dv, dw, ds])


@pytest.mark.parametrize("u", [-0.05, 0.06, 0.09, 0.2, 0.25, 0.4, 0.9087, 1.2, 1.5])
def test_bocf_reduces_to_sharp_model_away_from_thresholds(u):
    """All thresholds (0.006, 0.006, 0.13, 0.3) are > 1/(2k) = 0.0176 away from these u."""
    for (v, w, s) in [(0.9, 0.8, 0.1), (0.2, 0.95, 0.6)]:
        got = O.reaction(BOCF, [u, v, w, s])
        ref = _bocf_sharp(u, v, w, s)
        assert got == pytest.approx(ref, rel=1e-13, abs=1e-15)


def test_bocf_inside_transition_zone_closed_form():
    """u = 0 sits inside the k = 28.4 transition zone of theta_v^- = theta_o = 0.006 (Q10):
    v_inf = H(0.006), w_inf = (1 - H(-0.006)) + 0.94 H(-0.006), tau_v^- = 60 + 1090 H(-0.006)."""
    hp, hm = smoothstep(0.006), smoothstep(-0.006)
    v, w, s = 0.3, 0.5, 0.2
    f = O.reaction(BOCF, [0.0, v, w, s])
    assert f[0] == 0.0  # no current at u = u_o = 0 whatever the gates
    tvm = 60.0 + hm * (1150.0 - 60.0)
    assert f[1] == pytest.approx((hp - v) / tvm, rel=1e-13)
    twm = 60.0 + (15.0 - 60.0) * (1 + np.tanh(65.0 * (0.0 - 0.03))) / 2
    winf = (1 - hm) * 1.0 + hm * 0.94
    assert f[2] == pytest.approx((winf - w) / twm, rel=1e-13)
    assert f[3] == pytest.approx(((1 + np.tanh(2.0994 * (0.0 - 0.9087))) / 2 - s) / 2.7342, rel=1e-13)
    # rest state = (0, v_inf, w_inf, s_inf(0)), not (0,1,1,0)
    rest = np.array(W.REST[BOCF])
    assert rest == pytest.approx([0.0, hp, winf, (1 + np.tanh(-2.0994 * 0.9087)) / 2], abs=2e-15)
    assert np.max(np.abs(O.reaction(BOCF, rest))) < 1e-15


def test_bocf_single_cell_action_potential():
    """Peak u in the printed range (0, 1.55); action potential lasts ~270 ms (SURVEY.md A10:
    time above u = 0.13 is 270.8 ms for the 'H_k everywhere' reading)."""
    rest = np.array(W.REST[BOCF])
    z0 = rest.copy(); z0[0] = 0.5
    tr = _single_cell(BOCF, z0, 0.1, 4500)
    assert 1.3 < tr[:, 0].max() < GOLD["u_range"]["bocf"][1]
    assert tr[:, 0].min() > -1e-3
    assert np.all(tr[:, 1:] > -1e-9) and np.all(tr[:, 1:] < 1.0 + 1e-9)   # gates in (0,1)
    apd = 0.1 * np.count_nonzero(tr[:, 0] > 0.13)
    assert 255.0 < apd < 290.0, apd
    z0[0] = 0.2  # below theta_v = 0.3: no upstroke
    tr = _single_cell(BOCF, z0, 0.1, 1000)
    assert tr[:, 0].max() <= 0.2 + 1e-12 and tr[-1, 0] < 0.02


def test_tanhfree_variant_matches_slope_and_limits():
    """tanh(x) -> 2 H_k'(x) - 1; k' = 1/3 matches the unit slope at 0 and saturates
    at |x| >= 3/2."""
    # Karma: only the (1 - tanh(u - u_h)) factor changes
    f0 = O.reaction(KARMA, [3.0, 0.2], variant=0)
    f1 = O.reaction(KARMA, [3.0, 0.2], variant=1)
    assert f0 == pytest.approx(f1, abs=1e-15)          # tanh(0) = 2H(0) - 1 = 0
    f1 = O.reaction(KARMA, [1.0, 0.2], variant=1)      # u - u_h = -2 <= -3/2: factor (1 - (-1)) = 2
    assert f1[0] == pytest.approx((0.5 * 2.0 * (1.5415 - 0.2 ** 6) - 1.0) / 2.5, abs=1e-15)
    e = 1e-6
    d = (O.reaction(KARMA, [3.0 + e, 0.0], variant=1)[0] - O.reaction(KARMA, [3.0 - e, 0.0], variant=1)[0]) / (2 * e)
    d0 = (O.reaction(KARMA, [3.0 + e, 0.0], variant=0)[0] - O.reaction(KARMA, [3.0 - e, 0.0], variant=0)[0]) / (2 * e)
    assert d == pytest.approx(d0, rel=1e-6)
