"""B200-native index-based multi-walk force evaluation (arXiv 1907.02290, 'Accelerated FDPS').

`binding` wraps the C-ABI CUDA library (include/mwf.h); `workload` builds seeded synthetic inputs.
"""
__version__ = "0.1.0"
