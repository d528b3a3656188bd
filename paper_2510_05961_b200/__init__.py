"""B200-native multilevel summation (MSM) with B-spline interpolation: the energy / force /
potential / virial hot path of arxiv 2510.05961 behind a C-ABI library (include/msm.h).

`workloads` (seeded input generators) imports nothing else from this package; the CUDA binding
is loaded lazily by `paper_2510_05961_b200.msm`.
"""
__all__ = ["workloads"]
