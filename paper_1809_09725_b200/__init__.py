"""cp4d -- B200-native Chambolle-Pock iteration for time-decomposed 4D tomography (arXiv 1809.09725).

`synth` (seeded input generators) imports without a GPU; everything else goes through the C-ABI library
`libcp4d.so` (see include/cp4d.h) via `binding` (and `slabs`, the z-slab drivers on top of it), which raises if the CUDA library is missing -- there is
no CPU fallback.
"""
__all__ = ["synth", "binding", "build", "slabs"]
