"""B200-native (sm_100a, fp64) GAMER-SR hot path: C-ABI CUDA library + thin Python binding.

`workloads` (numpy only, seeded input generators) can be imported without CUDA; everything else
goes through `binding`, which dlopens the in-tree libsrhd_b200.so and fails loudly without it.
"""
from . import workloads  # noqa: F401

__all__ = ["workloads", "binding", "build", "driver"]
