"""B200-native Stokesian-dynamics mobility product (Kopp & Hoefling, arXiv:1205.6333).

`paper_1205_6333_b200.sd` is the thin Python binding of the C-ABI library `libsd_b200.so`
(include/sd_b200.h); `paper_1205_6333_b200.workloads` holds the seeded input generators.
Nothing is loaded at import time; the CUDA library is opened on first use and there is no
CPU fallback.
"""

__all__ = ["sd", "workloads"]
