"""B200-native primal-dual dipole deconvolution (hot path of arXiv 2006.09808).

The CUDA library is loaded lazily by `paper_2006_09808_b200.binding`; importing the package
(or `paper_2006_09808_b200.synth`, the seeded input generator) needs neither a GPU nor the
built extension.
"""
__all__ = ["binding", "shard", "synth"]
