"""paper_2002_00054_b200 -- B200-native (sm_100a) Behler-Parrinello NNP energy + force path.

The product is the C-ABI library `libnnp_b200.so` (include/nnp.h, sources in csrc/); this
package only marshals arguments for it (binding.py) and builds it (build.py).
"""
from .binding import EXPORTS, NNP, NNPError, STAGE_NAMES, load_library, measure_fp64_peak  # noqa: F401

__all__ = ["NNP", "NNPError", "load_library", "measure_fp64_peak", "EXPORTS", "STAGE_NAMES"]
