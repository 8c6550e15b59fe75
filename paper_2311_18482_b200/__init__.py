"""legs — B200-native hot path of Language Embedded 3D Gaussians (arxiv 2311.18482).

The CUDA library (csrc/ -> liblegs.so, C-ABI declared in include/legs.h) is loaded lazily by `binding`;
every compute entry point raises if the library is missing (there is no CPU fallback).
`inputs` holds the seeded synthetic input generators (no method arithmetic).
"""
__all__ = ["inputs", "binding", "build"]
