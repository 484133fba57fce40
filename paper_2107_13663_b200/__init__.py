"""paper_2107_13663_b200 -- thin Python binding of libm3dk (include/m3dk.h).

The energetic-particle push of M3D-C1-K (arXiv 2107.13663) for NVIDIA B200: slow-manifold Boris push + finite-element
field evaluation + delta-f weight, fused CUDA kernels behind a C ABI.  This module only marshals arguments: every step
of the hot path runs in the kernels of ``csrc/``.  PyTorch supplies device memory and the stream, nothing else.

There is no CPU fallback: without the compiled library or without a CUDA device every call raises.
"""
from __future__ import annotations

from ._binding import (  # noqa: F401
    M3DKError,
    Pusher,
    lib,
    lib_path,
    exported_symbols,
    F0_MAXWELLIAN,
    F0_SLOWING_DOWN,
    F0_BEAM_PITCH,
    STATE_KEYS,
)
from ._build import build, build_all  # noqa: F401
