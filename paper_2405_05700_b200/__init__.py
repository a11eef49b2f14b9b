"""B200-native Cherenkov photon propagation with batched submission (arXiv:2405.05700 hot path).

The CUDA library is loaded lazily by :mod:`paper_2405_05700_b200.binding`; importing the
package (or :mod:`.workloads`) never touches the GPU or the shared library.
"""
__all__ = ["workloads", "binding"]
