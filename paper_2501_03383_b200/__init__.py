"""B200-native far-field radiation detector (arXiv 2501.03383 hot path).

The CUDA library is loaded lazily by :mod:`paper_2501_03383_b200.binding`; importing the
package (e.g. for :mod:`workloads`) needs neither a GPU nor the built library.
"""
__all__ = ["workloads", "binding"]
