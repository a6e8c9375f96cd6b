"""fftb-b200: B200-native batched sphere <-> cuboid 3D FFT (hot path of arXiv 2406.05577).

Importing the package has no side effects; the CUDA library is loaded on first use of
``paper_2406_05577_b200.binding`` (and fails loudly if it has not been built).
"""
__all__ = ["binding", "workloads"]
