"""B200-native GANDALF KRMHD hot path (arXiv 2511.21891): pseudo-spectral RHS + integrating-factor step.

`paper_2511_21891_b200.gandalf` is the thin Python binding over the C-ABI library
(include/gandalf.h); `paper_2511_21891_b200.synth` holds the seeded input generators.
The CUDA library is loaded lazily by the binding and its absence is a hard error there.
"""
__all__ = ["synth", "gandalf"]
