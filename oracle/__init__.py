"""TEST INFRASTRUCTURE, NOT THE PRODUCT: the CPU oracle of the hot path (see cardiac_oracle.c).

Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may
import this package.  It imports nothing from paper_1309_1720_b200.
"""
from .oracle import (build, lib, num_fields, num_params, default_params, hk, reaction, laplacian,
                     rhs, step, jvp, scheme_bits, threads, laplacian3d, step3d, build_timing,
                     cpu_model)

__all__ = ["build", "lib", "num_fields", "num_params", "default_params", "hk", "reaction",
           "laplacian", "rhs", "step", "jvp", "scheme_bits", "threads", "laplacian3d", "step3d",
           "build_timing", "cpu_model"]
