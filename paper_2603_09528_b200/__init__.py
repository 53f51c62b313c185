"""B200 (sm_100a) tensor-product–Thomas Poisson/Helmholtz solver (arxiv/paper_2603_09528 hot path).

`api` is the thin Python binding of the C-ABI library (include/tpt.h); `inputs` holds the seeded
synthetic input generators; `build` compiles the library with nvcc.  There is no CPU fallback:
using `api` without the built CUDA library, or without a B200, raises.
"""
from . import inputs  # noqa: F401

__all__ = ["inputs", "api", "build"]
