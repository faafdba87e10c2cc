"""B200-native TILD particle-mesh force path (PAPER.md arxiv 2302.02474, MATILDA.FT, section IV.C).

`paper_2302_02474_b200.tild` is the thin ctypes binding over the C-ABI library (include/tild.h);
`paper_2302_02474_b200.inputs` holds the seeded synthetic input recipes.  Importing the package does
not load the CUDA library; `tild.load()` does and fails loudly when it is missing.
"""
__all__ = ["inputs", "tild"]
