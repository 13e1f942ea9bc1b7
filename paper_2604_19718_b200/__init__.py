"""B200-native inside pass / sampler for codon-constrained RNA design (arXiv 2604.19718 hot path).

`binding` wraps the C-ABI CUDA library (include/cdz.h); `inputs` holds the seeded synthetic generators.
"""
from . import inputs  # noqa: F401
