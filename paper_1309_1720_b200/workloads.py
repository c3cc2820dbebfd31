"""Seeded synthetic inputs for the five BASELINE.json configs and the size sweep.

This module is the ONLY code shared by the CUDA path and the oracle's tests: it produces plain
numpy float64 arrays (dense ``[batch][n_v][ny][nx]``, x fastest) that both sides consume.  It holds
none of the method's arithmetic: no model right-hand side, no integrator, no Laplacian of the
method.  (The block-noise recipe of config 3 blurs its random blocks with ten Jacobi-style
averaging sweeps — that is part of the INPUT recipe of BASELINE.json:configs[2], written here with
``numpy.pad(mode="reflect")``; neither the oracle nor the kernels are involved.)

The paper uses no dataset; grids, models, dx and parameters follow PAPER.md:54, :63, :76 and the
grid sizes of its Figs. 3 and 5.  The concrete initial states are the
readings of SURVEY.md §8(d) / DESIGN.md "Input recipe".

Random numbers: a counter-based generator (splitmix64 finaliser applied to ``seed*2^32 + counter``),
``uniform = (x >> 11) * 2^-53``, Gaussian by Box-Muller, drawn in flat-index order, field-major.
"""
from __future__ import annotations

from dataclasses import dataclass, replace
import numpy as np

# ----------------------------------------------------------------------------- constants
FHN, KARMA, BOCF = 0, 1, 2
LAP5, LAP9X4, BOX9 = 0, 1, 2
EULER, HEUN, RK4, RUSH_LARSEN, IMPLICIT_EULER = 0, 1, 2, 3, 4

MODEL_NAMES = {FHN: "fhn", KARMA: "karma", BOCF: "bocf"}
STENCIL_NAMES = {LAP5: "lap5", LAP9X4: "lap9x4", BOX9: "box9"}
INTEGRATOR_NAMES = {EULER: "euler", HEUN: "heun", RK4: "rk4", RUSH_LARSEN: "rush_larsen",
                    IMPLICIT_EULER: "implicit_euler"}
NUM_FIELDS = {FHN: 2, KARMA: 2, BOCF: 4}
NUM_DIFFUSING = {FHN: 2, KARMA: 1, BOCF: 1}
STAGES = {EULER: 1, HEUN: 2, RK4: 4, RUSH_LARSEN: 1, IMPLICIT_EULER: 1}
RADIUS = {LAP5: 1, LAP9X4: 2, BOX9: 1}

# grid spacing and the largest diffusion constant per model
# (FHN delta = 1.5; Karma gamma = 0.0011 cm^2/ms; BOCF D = 1.171 cm^2/s
# = 1.171e-3 cm^2/ms, Q9(ii)).
DX = {FHN: 0.04, KARMA: 0.0262, BOCF: 0.03}
D_MAX = {FHN: 1.5, KARMA: 0.0011, BOCF: 1.171e-3}

# voltage ranges printed at PAPER.md:96 (gates are in (0,1))
U_RANGE = {FHN: (-1.0, 1.0), KARMA: (0.0, 3.5), BOCF: (0.0, 1.55)}

# Rest states (fixed points of N[z] = 0 of the models as implemented, Q10).  Written by
# `python -m oracle.rest_states` (which calls only oracle/; BOCF u printed as 1.5e-38, entered as the
# exact fixed point 0) and pinned by tests/test_oracle_models.py.
REST = {
    FHN: (-0.6591465811607408, -0.37276438744049384),
    KARMA: (0.0, 0.0),
    BOCF: (0.0, 0.7457044766720001, 0.98474226860032, 0.021553043080280773),
}
# peak of the slow FHN variable along a single-cell excursion from (1, v_rest);
# config 2 sets "refractory = 0.5 of its range".
FHN_V_PEAK = 0.4165


def default_dt(model: int) -> float:
    """dt = 0.5 * dx^2 / (4 D_max) for every config (BASELINE.json:configs[0]; Q6)."""
    return 0.5 * DX[model] ** 2 / (4.0 * D_MAX[model])


# ----------------------------------------------------------------------------- RNG
_M64 = np.uint64(0xFFFFFFFFFFFFFFFF)


def _splitmix64(x: np.ndarray) -> np.ndarray:
    with np.errstate(over="ignore"):
        x = (x + np.uint64(0x9E3779B97F4A7C15)) & _M64
        z = x
        z = ((z ^ (z >> np.uint64(30))) * np.uint64(0xBF58476D1CE4E5B9)) & _M64
        z = ((z ^ (z >> np.uint64(27))) * np.uint64(0x94D049BB133111EB)) & _M64
        return z ^ (z >> np.uint64(31))


def uniform01(seed: int, n: int, stream: int = 0) -> np.ndarray:
    """n uniforms in [0,1): counter-based, reproducible and independent of chunking."""
    ctr = np.arange(n, dtype=np.uint64)
    key = _splitmix64(np.array([np.uint64(seed) * np.uint64(0x100000000) + np.uint64(stream)],
                               dtype=np.uint64))[0]
    with np.errstate(over="ignore"):
        x = _splitmix64(ctr ^ key)
    return (x >> np.uint64(11)).astype(np.float64) * (1.0 / 9007199254740992.0)


def gaussian(seed: int, n: int, stream: int = 0) -> np.ndarray:
    """n standard normals by Box-Muller from two uniform streams."""
    u1 = uniform01(seed, n, stream=2 * stream + 101)
    u2 = uniform01(seed, n, stream=2 * stream + 102)
    return np.sqrt(-2.0 * np.log(1.0 - u1)) * np.cos(2.0 * np.pi * u2)


# ----------------------------------------------------------------------------- configs
@dataclass(frozen=True)
class Config:
    name: str
    model: int
    nx: int
    ny: int
    stencil: int
    integrator: int
    nsteps: int
    batch: int = 1
    seed: int = 0
    dx: float = 0.0
    dt: float = 0.0
    boundary: int = 0   # 0 no-flux, 1 periodic
    variant: int = 0    # 0 as printed, 1 tanh-free
    nz: int = 1         # > 1: 3-D grid [nz][ny][nx] (DESIGN.md f4)

    @property
    def n_v(self) -> int:
        return NUM_FIELDS[self.model]

    @property
    def scheme(self) -> int:
        return self.stencil | (self.integrator << 8) | (self.boundary << 16) | (self.variant << 24)

    @property
    def cells(self) -> int:
        return self.nx * self.ny * self.nz * self.batch

    def describe(self) -> str:
        return (f"{self.name}: {MODEL_NAMES[self.model]} {self.batch}x{self.ny}x{self.nx} "
                f"{STENCIL_NAMES[self.stencil]} {INTEGRATOR_NAMES[self.integrator]} "
                f"{self.nsteps} steps")


def make_config(name, model, n, stencil, integrator, nsteps, batch=1, seed=0, ny=None, **kw) -> Config:
    return Config(name=name, model=model, nx=n, ny=n if ny is None else ny, stencil=stencil,
                  integrator=integrator, nsteps=nsteps, batch=batch, seed=seed,
                  dx=DX[model], dt=default_dt(model), **kw)


def baseline_config(i: int) -> Config:
    """The five configs of BASELINE.json (1-based)."""
    if i == 1:
        return make_config("cfg1", FHN, 64, LAP5, EULER, 200, seed=1)
    if i == 2:
        return make_config("cfg2", FHN, 512, LAP9X4, RK4, 10_000, seed=2)
    if i == 3:
        return make_config("cfg3", KARMA, 1024, LAP5, RK4, 5_000, seed=3)
    if i == 4:
        return make_config("cfg4", BOCF, 2048, LAP9X4, RK4, 2_000, seed=4)
    if i == 5:
        return make_config("cfg5", FHN, 512, LAP9X4, RK4, 1_000, batch=17, seed=5)
    raise ValueError("config index must be 1..5")


def scaled(cfg: Config, n: int, nsteps: int | None = None, ny: int | None = None) -> Config:
    """Same config on an n x n (or n x ny) grid, for oracle-sized parity cases."""
    return replace(cfg, nx=n, ny=n if ny is None else ny,
                   nsteps=cfg.nsteps if nsteps is None else nsteps,
                   name=f"{cfg.name}@{n}")


# ----------------------------------------------------------------------------- initial states
def _fields(cfg: Config) -> np.ndarray:
    z = np.empty((cfg.n_v, cfg.ny, cfg.nx), dtype=np.float64)
    for f, r in enumerate(REST[cfg.model]):
        z[f] = r
    return z


def state_cfg1(cfg: Config) -> np.ndarray:
    """u = 1 on the left 5 columns, rest elsewhere, + U(-1e-3, 1e-3) on every field."""
    z = _fields(cfg)
    z[0, :, :5] = 1.0
    n = z.size
    z += (2.0 * uniform01(cfg.seed, n).reshape(z.shape) - 1.0) * 1e-3
    return z[None]


def state_cfg2(cfg: Config, noise: float = 1e-6, seed: int | None = None) -> np.ndarray:
    """Cross-field stimulus: u excited in the lower-left quadrant, slow variable half-way to its
    peak in the upper half, + noise * N(0,1)."""
    z = _fields(cfg)
    hx, hy = cfg.nx // 2, cfg.ny // 2
    z[0, :hy, :hx] = 1.0
    v_rest = REST[FHN][1]
    z[1, hy:, :] = v_rest + 0.5 * (FHN_V_PEAK - v_rest)
    z += noise * gaussian(cfg.seed if seed is None else seed, z.size).reshape(z.shape)
    return z[None]


def _smooth(f: np.ndarray, sweeps: int) -> np.ndarray:
    for _ in range(sweeps):
        p = np.pad(f, 1, mode="reflect")
        f = f + 0.125 * (p[1:-1, 2:] + p[1:-1, :-2] + p[2:, 1:-1] + p[:-2, 1:-1] - 4.0 * f)
    return f


def state_blocks(cfg: Config, block: int = 16, sweeps: int = 10, seed: int | None = None) -> np.ndarray:
    """Config-3 recipe for any model: per block x block cells, u ~ U[u range], every other field
    ~ U[0,1] (FHN v ~ U[v_rest, v_peak]); then `sweeps` averaging sweeps per field."""
    seed = cfg.seed if seed is None else seed
    nbx, nby = -(-cfg.nx // block), -(-cfg.ny // block)
    z = np.empty((cfg.n_v, cfg.ny, cfg.nx), dtype=np.float64)
    for f in range(cfg.n_v):
        r = uniform01(seed, nbx * nby, stream=f).reshape(nby, nbx)
        if f == 0:
            lo, hi = U_RANGE[cfg.model]
            if cfg.model == FHN:
                lo = REST[FHN][0]
        elif cfg.model == FHN:
            lo, hi = REST[FHN][1], FHN_V_PEAK
        else:
            lo, hi = 0.0, 1.0
        coarse = lo + (hi - lo) * r
        fine = np.repeat(np.repeat(coarse, block, axis=0), block, axis=1)[:cfg.ny, :cfg.nx]
        z[f] = _smooth(np.ascontiguousarray(fine), sweeps)
    return z[None]


def state_cfg4(cfg: Config, strip: int = 8) -> np.ndarray:
    """Rest state everywhere, u = 1 on the left `strip` columns (planar wave)."""
    z = _fields(cfg)
    z[0, :, :strip] = 1.0
    return z[None]


def stimulus_cfg4(state: np.ndarray) -> np.ndarray:
    """Cross-field stimulus applied at step 500 of config 4: u = 1 on the lower half."""
    out = state.copy()
    ny = out.shape[-2]
    out[:, 0, : ny // 2, :] = 1.0
    return out


def stimulus_cfg4_inplace(state):
    """The same edit in place on a numpy array or a torch tensor (host or device): plain slice
    assignment, no arithmetic."""
    ny = state.shape[-2]
    state[:, 0, : ny // 2, :] = 1.0
    return state


def directions_cfg5(cfg: Config, nvec: int, seed: int | None = None) -> np.ndarray:
    """nvec Gaussian directions over all n_v*ny*nx entries, Euclidean norm 1 each."""
    seed = cfg.seed if seed is None else seed
    n = cfg.n_v * cfg.ny * cfg.nx
    v = np.empty((nvec, cfg.n_v, cfg.ny, cfg.nx), dtype=np.float64)
    for b in range(nvec):
        g = gaussian(seed, n, stream=b)
        v[b] = (g / np.sqrt(np.sum(g * g))).reshape(cfg.n_v, cfg.ny, cfg.nx)
    return v


def state_cfg5(cfg: Config, base: np.ndarray, eps: float = 1e-7) -> np.ndarray:
    """[batch] states: member 0 = base, member b = base + eps * v_b."""
    base = np.asarray(base, dtype=np.float64).reshape(cfg.n_v, cfg.ny, cfg.nx)
    z = np.repeat(base[None], cfg.batch, axis=0)
    z[1:] += eps * directions_cfg5(cfg, cfg.batch - 1)
    return z


CFG5_BASE_STEPS = 5_000


def base_recipe_cfg5(cfg: Config) -> tuple[Config, np.ndarray, int]:
    """What BASELINE.json:configs[4] defines the base of config 5 as: the config-2-shaped state
    (same grid as `cfg`, seed 2) after 5,000 RK4 steps.  Returns (single-member config, its initial
    state, number of steps); the CALLER integrates it — with the oracle in tests/ and in
    bench.py --impl reference, with the library in bench.py — because this module holds none of the
    method's arithmetic — and passes the result to initial_state(cfg, base=...)."""
    one = replace(cfg, batch=1, nsteps=CFG5_BASE_STEPS, name="cfg2" if "@" not in cfg.name else f"cfg2@{cfg.nx}",
                  seed=2)
    return one, state_cfg2(one), CFG5_BASE_STEPS


def synthetic_base_cfg5(cfg: Config) -> np.ndarray:
    """Stand-in for 'config-2 state after 5000 steps' for the SCALED parity cases only (cfg5@N, where
    running 5000 steps is not the point): the config-2 initial state blurred so it is smooth like an
    evolved state.  The full-size config 5 never uses it (initial_state insists on a real base)."""
    one = replace(cfg, batch=1)
    z = state_cfg2(one, noise=0.0)[0]
    for f in range(z.shape[0]):
        z[f] = _smooth(z[f], 20)
    z += 1e-3 * gaussian(cfg.seed + 1000, z.size).reshape(z.shape)
    return z


def sweep_sizes() -> list[int]:
    """Grid sizes of the size sweep 'S' of SURVEY.md §8(d): the paper's Fig. 5 sweep through
    N0 ~ 362 extended to streaming sizes."""
    return [64, 128, 256, 362, 512, 768, 1024, 2048, 4096, 8192]


def sweep_config(model: int, n: int, stencil: int | None = None, integrator: int = RK4) -> Config:
    if stencil is None:
        stencil = LAP5 if model == KARMA else LAP9X4          # the stencils of configs 2-4
    nsteps = max(8, min(200, (1 << 28) // (n * n) * 8))       # 200 steps up to 1024^2, fewer beyond
    return make_config(f"sweep{n}", model, n, stencil, integrator, nsteps, seed=9)


def sweep_state(cfg: Config, base: int = 256) -> np.ndarray:
    """Config-3-style block-noise state of a base x base grid, repeated
    periodically to cfg.nx x cfg.ny: generating 8192^2 x 4 fields block by block on the host would
    take longer than the measurement; the kernels' speed does not depend on the values."""
    b = min(base, cfg.nx, cfg.ny)
    small = state_blocks(replace(cfg, nx=b, ny=b, batch=1))
    ry, rx = -(-cfg.ny // b), -(-cfg.nx // b)
    z = np.tile(small, (cfg.batch, 1, ry, rx))[:, :, :cfg.ny, :cfg.nx]
    return np.ascontiguousarray(z)


def state_3d(cfg: Config) -> np.ndarray:
    """3-D input: the block-noise recipe of config 3 per plane (a different seed per plane), then five
    averaging sweeps along z with mirrored ends, dense [batch][n_v][nz][ny][nx]."""
    planes = [state_blocks(replace(cfg, nz=1, batch=1), seed=cfg.seed + 31 * k)[0] for k in range(cfg.nz)]
    z = np.stack(planes, axis=1)                     # [n_v][nz][ny][nx]
    for _ in range(5):
        p = np.pad(z, ((0, 0), (1, 1), (0, 0), (0, 0)), mode="reflect")
        z = 0.5 * z + 0.25 * (p[:, :-2] + p[:, 2:])
    out = np.repeat(z[None], cfg.batch, axis=0)
    if cfg.batch > 1:
        out[1:] += 1e-3 * gaussian(cfg.seed + 77, out[1:].size).reshape(out[1:].shape)
    return np.ascontiguousarray(out)


def default_dt_3d(model: int) -> float:
    """Half the explicit limit of the 7-point stencil, dx^2 / (6 D_max)."""
    return 0.5 * DX[model] ** 2 / (6.0 * D_MAX[model])


def initial_state(cfg: Config, base: np.ndarray | None = None) -> np.ndarray:
    """Initial state of a (possibly scaled) baseline config, dense [batch][n_v][ny][nx].
    Config 5 at full size needs `base`, the integrated state of base_recipe_cfg5()."""
    if cfg.nz > 1:
        return state_3d(cfg)
    name = cfg.name.split("@")[0]
    if name == "cfg1":
        return state_cfg1(cfg)
    if name == "cfg2":
        return state_cfg2(cfg)
    if name == "cfg3":
        return state_blocks(cfg)
    if name == "cfg4":
        return state_cfg4(cfg)
    if name == "cfg5":
        if base is None:
            if "@" not in cfg.name:
                raise ValueError("config 5 is defined on the config-2 state after 5000 RK4 steps: integrate "
                                 "base_recipe_cfg5(cfg) and pass it as base=")
            base = synthetic_base_cfg5(cfg)
        return state_cfg5(cfg, base)
    z = state_blocks(cfg)
    if cfg.batch > 1:
        z = np.repeat(z, cfg.batch, axis=0)
        z[1:] += 1e-3 * gaussian(cfg.seed + 77, z[1:].size).reshape(z[1:].shape)
    return z
