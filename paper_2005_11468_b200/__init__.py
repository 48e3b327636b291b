"""B200 (sm_100a) batched perfectly-stirred-reactor chemistry: the hot path of arxiv 2005.11468.

`synth` builds seeded inputs; `binding` is the thin ctypes layer over the C ABI in include/psr.h
(libpsr_b200.so, built from csrc/ by `build`).  Nothing here computes chemistry on the host.
"""
from . import synth  # noqa: F401  (pure numpy, importable without the CUDA library)

__all__ = ["synth", "binding", "build"]
