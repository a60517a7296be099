"""B200-native FDTD Yee update with a systolic, time-skewed schedule (arXiv 2502.20610).

`workloads` (seeded synthetic inputs) imports without the CUDA library; `binding` loads
`libfdtd_b200.so` on first use and fails loudly if it is missing -- there is no CPU fallback.
"""
__all__ = ["workloads", "binding"]
