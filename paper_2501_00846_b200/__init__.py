"""tslb-b200: B200-native TSLB + conservative Allen-Cahn hot path (arXiv 2501.00846).

`paper_2501_00846_b200.binding` is the thin Python layer over the C-ABI CUDA library
(include/tslb.h); `paper_2501_00846_b200.inputs` holds the seeded input generators.
"""
__all__ = ["inputs", "binding"]
