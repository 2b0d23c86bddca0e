"""b200-md: single-GPU MD hot path of Glaser et al. (arXiv:1412.3387) for NVIDIA B200 (sm_100a).

Importing this package loads nothing: `paper_1412_3387_b200.inputs` (seeded synthetic workloads, numpy
only) is usable without a GPU, and `paper_1412_3387_b200.binding` opens the C-ABI shared library
(`csrc/libb200md.so`) on first use and raises loudly if it is missing.  There is no CPU fallback.
"""

__all__ = ["inputs", "binding"]
