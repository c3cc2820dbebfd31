"""ctypes binding of libcardiac.so — same names as include/cardiac.h (and the diagnostics of
include/cardiac_diag.h, the allocation-free entry point of include/cardiac_static.h), argument marshalling only.

Every step of the hot path runs in the library's CUDA kernels; there is no CPU fallback here.
Importing this module fails loudly if the library has not been built
(``python -m paper_1309_1720_b200.build``), and every call that touches the device fails with
``CardiacError`` when no B200 is present.

State arguments may be numpy float64 arrays (host) or torch float64 tensors (host or CUDA);
``torch`` is used for device memory and streams only.
"""
from __future__ import annotations

import ctypes
import os

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(_HERE, "libcardiac.so")

# enums of include/cardiac.h
CARDIAC_FHN, CARDIAC_KARMA, CARDIAC_BOCF = 0, 1, 2
CARDIAC_LAP5, CARDIAC_LAP9X4, CARDIAC_BOX9 = 0, 1, 2
CARDIAC_EULER, CARDIAC_HEUN, CARDIAC_RK4 = 0 << 8, 1 << 8, 2 << 8
CARDIAC_RUSH_LARSEN, CARDIAC_IMPLICIT_EULER = 3 << 8, 4 << 8
CARDIAC_NOFLUX, CARDIAC_PERIODIC = 0 << 16, 1 << 16
CARDIAC_VARIANT_PAPER, CARDIAC_VARIANT_TANHFREE = 0 << 24, 1 << 24
CARDIAC_PLAN_AUTO, CARDIAC_PLAN_STAGE, CARDIAC_PLAN_FUSED, CARDIAC_PLAN_PERSISTENT, CARDIAC_PLAN_PAIR = 0, 1, 2, 3, 4
CARDIAC_PROBE_EXP, CARDIAC_PROBE_RCP, CARDIAC_PROBE_HK, CARDIAC_PROBE_REACTION = 0, 1, 2, 3
CARDIAC_OK, CARDIAC_ERR_INVALID, CARDIAC_ERR_CUDA, CARDIAC_ERR_NOSTATE, CARDIAC_ERR_WORKSPACE = 0, -1, -2, -3, -4

EXPORTS = [
    "cardiac_num_fields", "cardiac_num_params", "cardiac_default_params", "cardiac_create",
    "cardiac_create3d",    "cardiac_set_params", "cardiac_get_params", "cardiac_set_stream", "cardiac_set_plan",
    "cardiac_get_plan", "cardiac_workspace_bytes", "cardiac_bind_workspace", "cardiac_set_state",
    "cardiac_step", "cardiac_get_state", "cardiac_get_jvp", "cardiac_get_rows", "cardiac_set_rows",
    "cardiac_last_error", "cardiac_destroy",
]
# include/cardiac_diag.h: diagnostics for tests and bench.py, not part of the product boundary
DIAG_EXPORTS = ["cardiac_probe", "cardiac_launch_count", "cardiac_time_steps", "cardiac_measure_fp64_peak",
                "cardiac_measure_fp64_issue"]


# include/cardiac_static.h: the one entry point that allocates nothing (stage buffers in a static device array)
STATIC_EXPORTS = ["cardiac_step_static"]
CARDIAC_STATIC_SCRATCH_BYTES = 33554432


class CardiacError(RuntimeError):
    def __init__(self, code: int, message: str):
        super().__init__(f"libcardiac error {code}: {message}")
        self.code = code


if not os.path.exists(LIB_PATH):
    raise ImportError(f"{LIB_PATH} is missing: build it with `python -m paper_1309_1720_b200.build` "
                      "(there is no CPU fallback)")

_lib = ctypes.CDLL(LIB_PATH)
_vp, _dp, _i, _d, _ll = ctypes.c_void_p, ctypes.POINTER(ctypes.c_double), ctypes.c_int, ctypes.c_double, ctypes.c_longlong
_sig = {
    "cardiac_num_fields": (_i, [_i]),
    "cardiac_num_params": (_i, [_i]),
    "cardiac_default_params": (_i, [_i, _dp, _i]),
    "cardiac_create": (_vp, [_i, _i, _i, _d, _d, _i, _i]),
    "cardiac_create3d": (_vp, [_i, _i, _i, _i, _d, _d, _i, _i]),
    "cardiac_set_params": (_i, [_vp, _dp, _i]),
    "cardiac_get_params": (_i, [_vp, _dp, _i]),
    "cardiac_set_stream": (_i, [_vp, _vp]),
    "cardiac_set_plan": (_i, [_vp, _i, _i]),
    "cardiac_get_plan": (_i, [_vp]),
    "cardiac_workspace_bytes": (ctypes.c_size_t, [_vp]),
    "cardiac_bind_workspace": (_i, [_vp, _vp, ctypes.c_size_t]),
    "cardiac_set_state": (_i, [_vp, _vp, _i]),
    "cardiac_step": (_i, [_vp, _ll]),
    "cardiac_get_state": (_i, [_vp, _vp, _i]),
    "cardiac_get_jvp": (_i, [_vp, _d, _vp, _i]),
    "cardiac_get_rows": (_i, [_vp, _i, _i, _vp, _i]),
    "cardiac_set_rows": (_i, [_vp, _i, _i, _vp, _i]),
    "cardiac_probe": (_i, [_vp, _i, _vp, _vp, _ll]),
    "cardiac_launch_count": (_ll, [_vp]),
    "cardiac_time_steps": (_i, [_vp, _ll, _i, ctypes.POINTER(ctypes.c_float)]),
    "cardiac_measure_fp64_peak": (_i, [_vp, _i, _i, _dp]),
    "cardiac_measure_fp64_issue": (_i, [_vp, _i, _i, _i, _dp]),
    "cardiac_step_static": (_i, [_i, _i, _i, _i, _i, _d, _d, _dp, _i, _vp, _vp, _ll, _vp, ctypes.c_char_p, _i]),
    "cardiac_last_error": (ctypes.c_char_p, [_vp]),
    "cardiac_destroy": (None, [_vp]),
}
for _name, (_res, _args) in _sig.items():
    _f = getattr(_lib, _name)
    _f.restype, _f.argtypes = _res, _args


def _check(ctx, rc: int) -> None:
    if rc != CARDIAC_OK:
        raise CardiacError(rc, (_lib.cardiac_last_error(ctx) or b"").decode())


def _buffer(x):
    """(address, on_device, keepalive) of a float64 numpy array or torch tensor."""
    if isinstance(x, np.ndarray):
        if x.dtype != np.float64 or not x.flags["C_CONTIGUOUS"]:
            raise TypeError("state arrays must be C-contiguous float64")
        return x.ctypes.data, 0, x
    import torch
    if isinstance(x, torch.Tensor):
        if x.dtype != torch.float64 or not x.is_contiguous():
            raise TypeError("state tensors must be contiguous float64")
        return x.data_ptr(), int(x.is_cuda), x
    raise TypeError("expected a numpy array or a torch tensor")


# ----------------------------------------------------------------------------- same names as the C ABI
def cardiac_num_fields(model: int) -> int:
    return _lib.cardiac_num_fields(model)


def cardiac_num_params(model: int) -> int:
    return _lib.cardiac_num_params(model)


def cardiac_default_params(model: int) -> np.ndarray:
    n = cardiac_num_params(model)
    if n < 0:
        raise CardiacError(CARDIAC_ERR_INVALID, "unknown model")
    p = np.zeros(n)
    rc = _lib.cardiac_default_params(model, p.ctypes.data_as(_dp), n)
    if rc:
        raise CardiacError(rc, "cardiac_default_params")
    return p


def cardiac_create(model: int, nx: int, ny: int, dx: float, dt: float, scheme: int, batch: int = 1):
    ctx = _lib.cardiac_create(model, nx, ny, dx, dt, scheme, batch)
    if not ctx:
        raise CardiacError(CARDIAC_ERR_INVALID, (_lib.cardiac_last_error(None) or b"").decode())
    return ctx


def cardiac_create3d(model: int, nx: int, ny: int, nz: int, dx: float, dt: float, scheme: int, batch: int = 1):
    ctx = _lib.cardiac_create3d(model, nx, ny, nz, dx, dt, scheme, batch)
    if not ctx:
        raise CardiacError(CARDIAC_ERR_INVALID, (_lib.cardiac_last_error(None) or b"").decode())
    return ctx


def cardiac_set_params(ctx, p) -> None:
    p = np.ascontiguousarray(p, dtype=np.float64)
    _check(ctx, _lib.cardiac_set_params(ctx, p.ctypes.data_as(_dp), p.size))


def cardiac_get_params(ctx, n: int) -> np.ndarray:
    p = np.zeros(n)
    _check(ctx, _lib.cardiac_get_params(ctx, p.ctypes.data_as(_dp), n))
    return p


def cardiac_set_stream(ctx, cuda_stream: int) -> None:
    _check(ctx, _lib.cardiac_set_stream(ctx, cuda_stream))


def cardiac_set_plan(ctx, plan: int, param: int = 0) -> None:
    _check(ctx, _lib.cardiac_set_plan(ctx, plan, param))


def cardiac_get_plan(ctx) -> int:
    return _lib.cardiac_get_plan(ctx)


def cardiac_workspace_bytes(ctx) -> int:
    return _lib.cardiac_workspace_bytes(ctx)


def cardiac_bind_workspace(ctx, dev_ptr: int, nbytes: int) -> None:
    _check(ctx, _lib.cardiac_bind_workspace(ctx, dev_ptr, nbytes))


def cardiac_set_state(ctx, src) -> None:
    addr, dev, _keep = _buffer(src)
    _check(ctx, _lib.cardiac_set_state(ctx, addr, dev))


def cardiac_step(ctx, nsteps: int) -> None:
    _check(ctx, _lib.cardiac_step(ctx, nsteps))


def cardiac_get_state(ctx, dst) -> None:
    addr, dev, _keep = _buffer(dst)
    _check(ctx, _lib.cardiac_get_state(ctx, addr, dev))


def cardiac_get_jvp(ctx, eps: float, dst) -> None:
    addr, dev, _keep = _buffer(dst)
    _check(ctx, _lib.cardiac_get_jvp(ctx, eps, addr, dev))


def cardiac_get_rows(ctx, j0: int, nrows: int, dst) -> None:
    addr, dev, _keep = _buffer(dst)
    _check(ctx, _lib.cardiac_get_rows(ctx, j0, nrows, addr, dev))


def cardiac_set_rows(ctx, j0: int, nrows: int, src) -> None:
    addr, dev, _keep = _buffer(src)
    _check(ctx, _lib.cardiac_set_rows(ctx, j0, nrows, addr, dev))


def cardiac_probe(ctx, what: int, src, dst, n: int) -> None:
    a, da, _k1 = _buffer(src)
    b, db, _k2 = _buffer(dst)
    if not (da and db):
        raise TypeError("cardiac_probe takes device tensors")
    _check(ctx, _lib.cardiac_probe(ctx, what, a, b, n))


def cardiac_launch_count(ctx) -> int:
    return _lib.cardiac_launch_count(ctx)


def cardiac_time_steps(ctx, nsteps: int, reps: int = 1) -> float:
    ms = ctypes.c_float(0.0)
    _check(ctx, _lib.cardiac_time_steps(ctx, nsteps, reps, ctypes.byref(ms)))
    return float(ms.value)


def cardiac_measure_fp64_peak(ctx, iters: int = 2000, reps: int = 5) -> float:
    """Thread-level DFMA instructions per second of the context's device (include/cardiac_diag.h)."""
    v = ctypes.c_double(0.0)
    _check(ctx, _lib.cardiac_measure_fp64_peak(ctx, iters, reps, ctypes.byref(v)))
    return float(v.value)


def cardiac_measure_fp64_issue(ctx, int_per_dfma: int, iters: int = 4000, reps: int = 3) -> float:
    """Thread-level DFMA per second with int_per_dfma integer instructions between them (cardiac_diag.h)."""
    v = ctypes.c_double(0.0)
    _check(ctx, _lib.cardiac_measure_fp64_issue(ctx, iters, reps, int_per_dfma, ctypes.byref(v)))
    return float(v.value)


def cardiac_step_static(model: int, scheme: int, nx: int, ny: int, batch: int, dx: float, dt: float, params,
                        src, dst, nsteps: int, cuda_stream: int = 0) -> None:
    """include/cardiac_static.h: `nsteps` time steps from the dense device state `src` into `dst` with the
    stage buffers in the library's static device array (no allocation; at most CARDIAC_STATIC_SCRATCH_BYTES)."""
    a_src, dev_src, _k1 = _buffer(src)
    a_dst, dev_dst, _k2 = _buffer(dst)
    if not (dev_src and dev_dst):
        raise TypeError("cardiac_step_static takes device tensors")
    if params is None:
        pp, npar = None, 0
    else:
        arr = np.ascontiguousarray(params, dtype=np.float64)
        pp, npar = arr.ctypes.data_as(_dp), int(arr.size)
    err = ctypes.create_string_buffer(512)
    rc = _lib.cardiac_step_static(model, scheme, nx, ny, batch, dx, dt, pp, npar, a_src, a_dst, nsteps,
                                  cuda_stream or None, err, len(err))
    if rc != CARDIAC_OK:
        raise CardiacError(rc, err.value.decode())


def cardiac_last_error(ctx=None) -> str:
    return (_lib.cardiac_last_error(ctx) or b"").decode()


def cardiac_destroy(ctx) -> None:
    _lib.cardiac_destroy(ctx)


# ----------------------------------------------------------------------------- convenience (marshalling only)
class Context:
    """RAII holder of a cardiac_ctx; torch provides the workspace memory and the stream."""

    def __init__(self, model, nx, ny, dx, dt, scheme, batch=1, plan=CARDIAC_PLAN_AUTO, plan_param=0,
                 params=None, use_torch_memory=True, nz=1):
        nv = cardiac_num_fields(model)
        self.shape = (batch, nv, ny, nx) if nz == 1 else (batch, nv, nz, ny, nx)
        self.ctx = (cardiac_create(model, nx, ny, dx, dt, scheme, batch) if nz == 1 else
                    cardiac_create3d(model, nx, ny, nz, dx, dt, scheme, batch))
        self._ws = None
        try:
            if params is not None:
                cardiac_set_params(self.ctx, params)
            if plan != CARDIAC_PLAN_AUTO or plan_param:
                cardiac_set_plan(self.ctx, plan, plan_param)
            if use_torch_memory:
                import torch
                nbytes = cardiac_workspace_bytes(self.ctx)
                self._ws = torch.empty(nbytes + 256, dtype=torch.uint8, device="cuda")
                ptr = (self._ws.data_ptr() + 255) // 256 * 256
                cardiac_bind_workspace(self.ctx, ptr, nbytes)
                cardiac_set_stream(self.ctx, torch.cuda.current_stream().cuda_stream)
        except Exception:
            cardiac_destroy(self.ctx)
            self.ctx = None
            raise

    @classmethod
    def from_config(cls, cfg, **kw):
        return cls(cfg.model, cfg.nx, cfg.ny, cfg.dx, cfg.dt, cfg.scheme, cfg.batch, nz=getattr(cfg, "nz", 1), **kw)

    def set_state(self, src):
        cardiac_set_state(self.ctx, src)

    def step(self, nsteps):
        cardiac_step(self.ctx, nsteps)

    def get_state(self, dst=None):
        if dst is None:
            dst = np.empty(self.shape, dtype=np.float64)
        cardiac_get_state(self.ctx, dst)
        return dst

    def get_rows(self, j0, nrows, dst=None):
        """Rows [j0, j0+nrows) of every field and member as dense [batch][n_v][nrows][nx]."""
        if dst is None:
            dst = np.empty(self.shape[:2] + (nrows, self.shape[-1]), dtype=np.float64)
        cardiac_get_rows(self.ctx, j0, nrows, dst)
        return dst

    def set_rows(self, j0, src):
        cardiac_set_rows(self.ctx, j0, src.shape[-2], src)

    def get_jvp(self, eps, dst=None):
        if dst is None:
            dst = np.empty((self.shape[0] - 1,) + self.shape[1:], dtype=np.float64)
        cardiac_get_jvp(self.ctx, eps, dst)
        return dst

    @property
    def launches(self):
        return cardiac_launch_count(self.ctx)

    @property
    def plan(self):
        return cardiac_get_plan(self.ctx)

    def close(self):
        if self.ctx:
            cardiac_destroy(self.ctx)
            self.ctx = None

    def __enter__(self):
        return self

    def __exit__(self, *exc):
        self.close()

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass
