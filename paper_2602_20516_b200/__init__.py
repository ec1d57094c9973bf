"""B200-native HMC molecular-dynamics force for SU(3) lattice gauge theory.

`paper_2602_20516_b200.lgt` is the thin Python binding over the C-ABI CUDA library
(include/lgt.h); `paper_2602_20516_b200.synth` makes the seeded synthetic inputs.
The binding is imported lazily so that `synth` stays usable without the CUDA library.
"""
__all__ = ["synth", "lgt"]
