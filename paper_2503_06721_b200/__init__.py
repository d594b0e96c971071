"""B200-native Wilson-Dirac operator for higher representations of SU(N) (arXiv 2503.06721, HiRep v2 hot path).

The CUDA library is loaded lazily by `paper_2503_06721_b200.hirep`; importing this package never
needs a GPU.  There is no CPU fallback: every operator call fails loudly if the CUDA library is missing.
"""
