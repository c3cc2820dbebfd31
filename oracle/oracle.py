"""ctypes binding of oracle/cardiac_oracle.c (test infrastructure; argument marshalling only)."""
from __future__ import annotations

import ctypes
import os
import subprocess
import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "cardiac_oracle.c")
_LIBS = {False: os.path.join(_HERE, "liboracle.so"), True: os.path.join(_HERE, "liboracle_omp.so")}
# the same source for TIMING only (bench.py's cpu_baseline / --impl reference): -O3 -march=native, which
# lets gcc contract and vectorise; never used for parity (SURVEY.md 8(d) "Oracle timing")
_TIMING_LIBS = {False: os.path.join(_HERE, "liboracle_fast.so"), True: os.path.join(_HERE, "liboracle_fast_omp.so")}
_loaded: dict = {}

_dp = ctypes.POINTER(ctypes.c_double)


def build(force: bool = False) -> None:
    """Compile the oracle: parity build (-O2 -ffp-contract=off, single thread) and the same source
    with -fopenmp (independent row loops split over threads, identical arithmetic)."""
    for omp, path in _LIBS.items():
        if not force and os.path.exists(path) and os.path.getmtime(path) >= os.path.getmtime(_SRC):
            continue
        cmd = ["gcc", "-O2", "-ffp-contract=off", "-fno-fast-math", "-shared", "-fPIC", "-o", path, _SRC, "-lm"]
        if omp:
            cmd.insert(1, "-fopenmp")
        subprocess.run(cmd, check=True)


def build_timing() -> None:
    """The timing build, compiled ON THE MACHINE THAT RUNS IT (-march=native): always rebuilt when the
    marker of this host is missing, so a library built on another CPU model never travels."""
    marker = os.path.join(_HERE, ".timing_host")
    host = _cpu_model()
    fresh = os.path.exists(marker) and open(marker).read() == host
    for omp, path in _TIMING_LIBS.items():
        if fresh and os.path.exists(path) and os.path.getmtime(path) >= os.path.getmtime(_SRC):
            continue
        cmd = ["gcc", "-O3", "-march=native", "-shared", "-fPIC", "-o", path, _SRC, "-lm"]
        if omp:
            cmd.insert(1, "-fopenmp")
        subprocess.run(cmd, check=True)
    with open(marker, "w") as fh:
        fh.write(host)


def _cpu_model() -> str:
    try:
        for line in open("/proc/cpuinfo"):
            if line.startswith("model name"):
                return line.split(":", 1)[1].strip()
    except OSError:
        pass
    return "unknown"


def cpu_model() -> str:
    return _cpu_model()


def lib(omp: bool = False, timing: bool = False) -> ctypes.CDLL:
    key = (omp, timing)
    if key not in _loaded:
        if timing:
            build_timing()
        else:
            build()
        L = ctypes.CDLL((_TIMING_LIBS if timing else _LIBS)[omp])
        L.oracle_num_fields.argtypes = [ctypes.c_int]
        L.oracle_num_params.argtypes = [ctypes.c_int]
        L.oracle_default_params.argtypes = [ctypes.c_int, _dp]
        L.oracle_hk.argtypes = [ctypes.c_double, ctypes.c_double]
        L.oracle_hk.restype = ctypes.c_double
        L.oracle_reaction.argtypes = [ctypes.c_int, ctypes.c_int, _dp, _dp, _dp]
        L.oracle_laplacian.argtypes = [_dp, _dp, ctypes.c_int, ctypes.c_int, ctypes.c_double,
                                       ctypes.c_int, ctypes.c_int]
        L.oracle_rhs.argtypes = [ctypes.c_int, ctypes.c_int, ctypes.c_int, ctypes.c_double,
                                 ctypes.c_int, _dp, _dp, _dp]
        L.oracle_step.argtypes = [ctypes.c_int, ctypes.c_int, ctypes.c_int, ctypes.c_double,
                                  ctypes.c_double, ctypes.c_int, ctypes.c_int, _dp, _dp,
                                  ctypes.c_longlong]
        L.oracle_laplacian3d.argtypes = [_dp, _dp, ctypes.c_int, ctypes.c_int, ctypes.c_int, ctypes.c_double,
                                         ctypes.c_int, ctypes.c_int]
        L.oracle_step3d.argtypes = [ctypes.c_int, ctypes.c_int, ctypes.c_int, ctypes.c_int, ctypes.c_double,
                                    ctypes.c_double, ctypes.c_int, ctypes.c_int, _dp, _dp,
                                    ctypes.c_longlong]
        L.oracle_jvp.argtypes = [_dp, ctypes.c_int, ctypes.c_size_t, ctypes.c_double, _dp]
        _loaded[key] = L
    return _loaded[key]


def threads(omp: bool) -> int:
    """Threads the chosen build uses."""
    if not omp:
        return 1
    env = os.environ.get("OMP_NUM_THREADS")
    return int(env) if env else (os.cpu_count() or 1)


def _ptr(a: np.ndarray):
    return a.ctypes.data_as(_dp)


def _c(a) -> np.ndarray:
    return np.ascontiguousarray(a, dtype=np.float64)


def scheme_bits(stencil=0, integrator=0, boundary=0, variant=0) -> int:
    return stencil | (integrator << 8) | (boundary << 16) | (variant << 24)


def num_fields(model: int) -> int:
    return lib().oracle_num_fields(model)


def num_params(model: int) -> int:
    return lib().oracle_num_params(model)


def default_params(model: int) -> np.ndarray:
    p = np.zeros(num_params(model))
    lib().oracle_default_params(model, _ptr(p))
    return p


def hk(x: float, k: float = 28.4) -> float:
    return lib().oracle_hk(float(x), float(k))


def reaction(model: int, z, params=None, variant: int = 0) -> np.ndarray:
    z = _c(z)
    p = default_params(model) if params is None else _c(params)
    f = np.zeros(num_fields(model))
    rc = lib().oracle_reaction(model, variant, _ptr(p), _ptr(z), _ptr(f))
    if rc:
        raise ValueError("oracle_reaction failed")
    return f


def laplacian(U, dx: float, stencil: int, boundary: int = 0) -> np.ndarray:
    U = _c(U)
    ny, nx = U.shape
    L = np.empty_like(U)
    rc = lib().oracle_laplacian(_ptr(U), _ptr(L), nx, ny, float(dx), stencil, boundary)
    if rc:
        raise ValueError("oracle_laplacian: invalid arguments")
    return L


def laplacian3d(U, dx: float, stencil: int, boundary: int = 0) -> np.ndarray:
    """3-D Laplacian of U[nz][ny][nx] (7-point for stencil 0, 13-point 4th-order cross for stencil 1)."""
    U = _c(U)
    nz, ny, nx = U.shape
    L = np.empty_like(U)
    rc = lib().oracle_laplacian3d(_ptr(U), _ptr(L), nx, ny, nz, float(dx), stencil, boundary)
    if rc:
        raise ValueError("oracle_laplacian3d: invalid arguments")
    return L


def step3d(model: int, Z, dx: float, dt: float, scheme: int, nsteps: int, params=None,
           omp: bool = False) -> np.ndarray:
    """Advance Z ([batch][n_v][nz][ny][nx] or [n_v][nz][ny][nx]) by nsteps; returns a new array."""
    Z = np.array(Z, dtype=np.float64, order="C", copy=True)
    shape = Z.shape
    if Z.ndim == 4:
        Z = Z[None]
    batch, nv, nz, ny, nx = Z.shape
    if nv != num_fields(model):
        raise ValueError("wrong number of fields")
    p = None if params is None else _c(params)
    rc = lib(omp).oracle_step3d(model, nx, ny, nz, float(dx), float(dt), scheme, batch,
                                None if p is None else _ptr(p), _ptr(Z), int(nsteps))
    if rc:
        raise ValueError(f"oracle_step3d failed ({rc})")
    return Z.reshape(shape)


def rhs(model: int, Z, dx: float, scheme: int, params=None) -> np.ndarray:
    Z = _c(Z)
    nv, ny, nx = Z.shape
    F = np.empty_like(Z)
    p = None if params is None else _c(params)
    rc = lib().oracle_rhs(model, nx, ny, float(dx), scheme, None if p is None else _ptr(p),
                          _ptr(Z), _ptr(F))
    if rc:
        raise ValueError("oracle_rhs failed")
    return F


def step(model: int, Z, dx: float, dt: float, scheme: int, nsteps: int, params=None,
         omp: bool = False, timing: bool = False) -> np.ndarray:
    """Advance Z ([batch][n_v][ny][nx] or [n_v][ny][nx]) by nsteps; returns a new array.
    timing=True runs the -O3 -march=native build (bench.py only; never for parity)."""
    Z = np.array(Z, dtype=np.float64, order="C", copy=True)
    shape = Z.shape
    if Z.ndim == 3:
        Z = Z[None]
    batch, nv, ny, nx = Z.shape
    if nv != num_fields(model):
        raise ValueError("wrong number of fields")
    p = None if params is None else _c(params)
    rc = lib(omp, timing).oracle_step(model, nx, ny, float(dx), float(dt), scheme, batch,
                              None if p is None else _ptr(p), _ptr(Z), int(nsteps))
    if rc:
        raise ValueError(f"oracle_step failed ({rc})")
    return Z.reshape(shape)


def jvp(Z, eps: float) -> np.ndarray:
    Z = _c(Z)
    batch = Z.shape[0]
    N = Z[0].size
    J = np.empty((batch - 1,) + Z.shape[1:])
    rc = lib().oracle_jvp(_ptr(Z), batch, N, float(eps), _ptr(J))
    if rc:
        raise ValueError("oracle_jvp failed")
    return J
