"""B200-native Monte-Carlo integrator for subtracted QED vertex graphs (arXiv:1909.08015 hot path).

The CUDA library is loaded lazily by `paper_1909_08015_b200.fg`; importing the package (or its
`inputs` module) does not need it.
"""
