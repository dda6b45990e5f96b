"""hfft: B200-native hybrid-FFT demagnetization field (arXiv 1910.07054).

``paper_1910_07054_b200.binding`` is the thin ctypes binding over the C-ABI library
(include/hfft.h); ``paper_1910_07054_b200.workloads`` holds the seeded input generators.
Nothing is imported eagerly so that the workloads can be used on a box without CUDA.
"""
__all__ = ["binding", "workloads"]
