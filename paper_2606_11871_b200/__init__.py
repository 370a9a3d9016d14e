"""WarpGuard protected-site CFI check engine, B200-native (arxiv/paper_2606_11871).

`binding`  thin ctypes face of the C-ABI library (include/warpguard.h); every step runs in CUDA.
`streams`  seeded synthetic policies / event streams (no method arithmetic).
"""
from . import streams  # noqa: F401

__all__ = ["streams"]
