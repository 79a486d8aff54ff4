"""krp: B200-native polarized Monte-Carlo radiative transfer hot path (arxiv 2512.01283).

`paper_2512_01283_b200.krp` is the thin ctypes binding of the C-ABI CUDA library declared in
include/krp.h (argument marshalling only); `paper_2512_01283_b200.inputs` holds the seeded
synthetic workloads (no arithmetic of the method).  Importing the package loads nothing; the
library is loaded on first use and its absence is an error, never a fallback.
"""
__all__ = ["krp", "inputs"]
