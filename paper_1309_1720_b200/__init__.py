"""paper_1309_1720_b200 — B200-native (sm_100a) explicit FP64 time stepping of cardiac
reaction-diffusion models (Marcotte & Grigoriev, arxiv 1309.1720).

The product is the C-ABI library ``libcardiac.so`` (include/cardiac.h); ``cardiac`` is its thin
ctypes binding (argument marshalling only) and ``workloads`` the seeded synthetic inputs.
"""
from . import workloads  # noqa: F401

__all__ = ["workloads", "cardiac"]


def __getattr__(name):
    if name == "cardiac":
        import importlib
        return importlib.import_module(".cardiac", __name__)
    raise AttributeError(name)
