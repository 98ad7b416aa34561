"""paper_1309_1894_b200 -- B200-native autotuned fp64 CSR SpMV (arxiv 1309.1894 method).

The CUDA library (csrc/ -> libspmv_b200.so) is loaded lazily by `binding`; importing
`workloads` (numpy-only input generators) does not need it.
"""
__version__ = "0.1.0"
