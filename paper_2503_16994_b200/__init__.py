"""paper_2503_16994_b200 -- B200-native clover Wilson-Dirac operator and CG propagator solve.

The CUDA library is loaded lazily by `paper_2503_16994_b200.binding` (importing this package or
`paper_2503_16994_b200.synth` never touches it, so CPU-only tools can use the input generators).
"""
__all__ = ["binding", "synth"]
