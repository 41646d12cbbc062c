"""B200-native hot path of the LOFAR lunar-pulse trigger pipeline (arXiv 1612.06592).

`paper_1612_06592_b200.binding` is the thin ctypes layer over the C-ABI library
(include/lofar_moon.h); `paper_1612_06592_b200.synth` the seeded input generator.
Importing the package does not load the CUDA library; `binding.load()` does and fails loudly
if it is missing.
"""
__all__ = ["binding", "synth", "build"]
