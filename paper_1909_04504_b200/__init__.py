"""B200-native SPH hot path (NNPS + pair loops + predictor-corrector) of arXiv 1909.04504.

Layout:
  workloads  -- seeded synthetic input generators (no SPH arithmetic; shared by tests/bench/oracle callers)
  binding    -- thin ctypes binding over the C-ABI library declared in include/sph.h
  build      -- in-tree nvcc build of csrc/*.cu -> libsph_b200.so

Nothing here falls back to the CPU: `binding` raises if the CUDA library is missing.
"""

__all__ = ["workloads", "binding", "build"]
