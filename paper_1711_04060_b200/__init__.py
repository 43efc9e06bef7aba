"""paper_1711_04060_b200 -- B200-native hot path of the GPU Poisson-Fermi solver of arXiv 1711.04060.

`pf`        : ctypes binding of the C ABI (include/pf.h) -> libpf_b200.so (hand-written CUDA, sm_100a)
`workloads` : seeded synthetic inputs for the BASELINE.json configs (no method arithmetic)
`build`     : in-tree nvcc build of the library
"""
__all__ = ["pf", "workloads", "build"]
