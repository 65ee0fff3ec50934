"""B200-native hot path of column-generation direct aperture optimization (arXiv 1003.5402).

The CUDA library is loaded lazily by :mod:`paper_1003_5402_b200.dao`; importing this package
(e.g. for the input generator) does not touch CUDA.
"""
__all__ = ["dao", "inputs"]
