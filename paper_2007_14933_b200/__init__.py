"""osbli-b200: B200-native residual + RK3 hot path of OpenSBLI (arXiv 2007.14933).

`paper_2007_14933_b200.osbli` is the thin ctypes binding of the C-ABI library
(include/osbli.h); `paper_2007_14933_b200.workloads` holds the seeded input generators.
There is no CPU fallback: importing `.osbli` raises if libosbli.so has not been built.
"""
__all__ = ["workloads"]
