"""B200-native causal-set action path (arXiv:1805.04463, Ch. 2-4).

Public API (argument marshalling only; every step runs in the CUDA kernels
behind the C ABI declared in include/causalset.h):

    from paper_1805_04463_b200 import api
    api.causal_matrix(coords, geometry)      -> (bits, bitsT)
    api.interval_hist(bits, bitsT, N, kmax)  -> hist (int64)
    api.bd_action(hist, N, dim)              -> S (fp64)

`inputs` holds the seeded synthetic sprinklers shared with the tests.
The CUDA library is loaded on first use of `api`; there is no CPU fallback.
"""
from . import inputs  # noqa: F401

__all__ = ["inputs", "api", "build"]


def __getattr__(name):
    if name in ("api", "build"):
        import importlib
        return importlib.import_module("." + name, __name__)
    raise AttributeError(name)
