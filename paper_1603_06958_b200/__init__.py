"""paper_1603_06958_b200 -- B200-native FAMSA stage I: all-pairs bit-parallel LCS similarity.

The product is the C-ABI library built from csrc/ (include/famsa_lcs.h) and the thin
binding in famsa.py.  `synth` is the shared seeded input generator.  There is no CPU
fallback: importing famsa without the built library raises.
"""
__all__ = ["famsa", "synth"]
