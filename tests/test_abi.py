"""The C-ABI library loads and exports every symbol include/cardiac.h declares; host-only entry
points behave; device entry points fail loudly without a GPU (no CPU fallback).  No GPU needed."""
import ctypes
import os
import re

import numpy as np
import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def C():
    from paper_1309_1720_b200 import build
    build.build()
    from paper_1309_1720_b200 import cardiac
    return cardiac


def _declared_functions(header="cardiac.h"):
    src = open(os.path.join(ROOT, "include", header)).read()
    src = re.sub(r"/\*.*?\*/", "", src, flags=re.S)
    return sorted(set(re.findall(r"\b(cardiac_[a-z0-9_]+)\s*\(", src)))


def test_every_declared_symbol_is_exported(C):
    names = _declared_functions()
    assert len(names) >= 15
    lib = ctypes.CDLL(C.LIB_PATH)
    for n in names:
        assert hasattr(lib, n), f"{n} declared in include/cardiac.h but not exported"
    assert sorted(C.EXPORTS) == names           # the binding covers exactly the header
    for n in names:
        assert callable(getattr(C, n))          # same names in Python
    # the diagnostics live in their own header (not part of the product boundary) and are covered likewise
    diag = _declared_functions("cardiac_diag.h")
    assert diag and not set(diag) & set(names)
    assert sorted(C.DIAG_EXPORTS) == diag
    for n in diag:
        assert hasattr(lib, n) and callable(getattr(C, n))
    assert not any(n in names for n in ("cardiac_probe", "cardiac_time_steps", "cardiac_launch_count"))
    # ... and so does the allocation-free entry point (include/cardiac_static.h)
    static = _declared_functions("cardiac_static.h")
    assert static == sorted(C.STATIC_EXPORTS) == ["cardiac_step_static"]
    assert hasattr(lib, static[0]) and callable(getattr(C, static[0]))
    src = open(os.path.join(ROOT, "include", "cardiac_static.h")).read()
    assert int(re.search(r"#define CARDIAC_STATIC_SCRATCH_BYTES (\d+)", src).group(1)) == C.CARDIAC_STATIC_SCRATCH_BYTES


def test_model_tables_and_defaults_agree_with_oracle(C):
    import oracle as O
    for m in (0, 1, 2):
        assert C.cardiac_num_fields(m) == O.num_fields(m)
        assert C.cardiac_num_params(m) == O.num_params(m)
        # typed independently on both sides; they must still be the same numbers
        assert np.array_equal(C.cardiac_default_params(m), O.default_params(m))
    assert C.cardiac_num_fields(9) == -1 and C.cardiac_num_params(-1) == -1


def test_enums_match_header(C):
    src = open(os.path.join(ROOT, "include", "cardiac.h")).read()
    for name in ("CARDIAC_FHN", "CARDIAC_KARMA", "CARDIAC_BOCF", "CARDIAC_LAP5", "CARDIAC_LAP9X4",
                 "CARDIAC_BOX9", "CARDIAC_PLAN_AUTO", "CARDIAC_PLAN_STAGE", "CARDIAC_PLAN_FUSED",
                 "CARDIAC_PLAN_PERSISTENT", "CARDIAC_PLAN_PAIR", "CARDIAC_OK", "CARDIAC_ERR_INVALID", "CARDIAC_ERR_CUDA",
                 "CARDIAC_ERR_NOSTATE", "CARDIAC_ERR_WORKSPACE"):
        m = re.search(rf"\b{name}\s*=\s*(-?\d+)", src)
        assert m and int(m.group(1)) == getattr(C, name), name
    for name in ("CARDIAC_EULER", "CARDIAC_HEUN", "CARDIAC_RK4", "CARDIAC_RUSH_LARSEN",
                 "CARDIAC_IMPLICIT_EULER", "CARDIAC_NOFLUX", "CARDIAC_PERIODIC",
                 "CARDIAC_VARIANT_PAPER", "CARDIAC_VARIANT_TANHFREE"):
        m = re.search(rf"\b{name}\s*=\s*(\d+)\s*<<\s*(\d+)", src)
        assert m and (int(m.group(1)) << int(m.group(2))) == getattr(C, name), name


def test_create_validates_before_touching_the_device(C):
    bad = [
        dict(model=5), dict(nx=2), dict(ny=2), dict(dx=0.0), dict(dx=float("inf")), dict(dt=-1.0),
        dict(dt=float("nan")), dict(batch=0), dict(scheme=7), dict(scheme=9 << 8),
        dict(scheme=C.CARDIAC_RUSH_LARSEN),              # gate integrators are BOCF-only
        dict(scheme=C.CARDIAC_LAP9X4, nx=4),             # needs >= 2r+1 = 5
        dict(scheme=3 << 16), dict(scheme=2 << 24),
    ]
    for kw in bad:
        a = dict(model=0, nx=16, ny=16, dx=0.04, dt=1e-4, scheme=0, batch=1)
        a.update(kw)
        with pytest.raises(C.CardiacError) as ei:
            C.cardiac_create(**a)
        assert "CUDA" not in str(ei.value), (kw, str(ei.value))   # rejected by validation, not by the driver
    assert C.cardiac_last_error(None) != ""


def test_null_context_is_rejected(C):
    assert C._lib.cardiac_step(None, 1) == C.CARDIAC_ERR_INVALID
    assert C._lib.cardiac_get_plan(None) == C.CARDIAC_ERR_INVALID
    assert C._lib.cardiac_workspace_bytes(None) == 0
    C._lib.cardiac_destroy(None)   # no-op


def test_no_cpu_fallback(C):
    """Without a usable B200 create() must fail (CUDA error text), never compute on the host."""
    import torch
    if torch.cuda.is_available():
        pytest.skip("GPU present: covered by the gpu tests")
    with pytest.raises(C.CardiacError) as ei:
        C.cardiac_create(0, 16, 16, 0.04, 1e-4, 0, 1)
    assert "CUDA" in str(ei.value) or "device" in str(ei.value)


def test_product_does_not_import_the_oracle():
    """The product path may not route through oracle/ (and vice versa)."""
    pkg = os.path.join(ROOT, "paper_1309_1720_b200")
    for dirpath, _, files in os.walk(pkg):
        for f in files:
            if f.endswith((".py", ".cu", ".cuh", ".h")):
                txt = open(os.path.join(dirpath, f)).read()
                assert not re.search(r"^\s*(from|import)\s+oracle\b", txt, flags=re.M), f
                assert "cardiac_oracle" not in txt and "liboracle" not in txt, f
    for f in os.listdir(os.path.join(ROOT, "oracle")):
        if f.endswith((".py", ".c")):
            txt = open(os.path.join(ROOT, "oracle", f)).read()
            assert "paper_1309_1720_b200 import" not in txt and "libcardiac" not in txt, f
