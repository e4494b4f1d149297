"""B200-native batched Kalman-filter track fitting and building (arxiv 1711.06571 hot path).

`synth` holds the seeded input generators (no KF arithmetic).  `binding` is the thin ctypes layer over the
C-ABI library `libkf_b200.so` (include/kf.h); it is imported lazily so that the generators can be used on a
machine without the CUDA build.
"""
__all__ = ["synth", "binding"]
