"""GSRQ encoder / decode hot path for NVIDIA B200 (sm_100a).

The product is the C-ABI library declared in include/gsrq.h (CUDA kernels under csrc/);
`paper_2607_01065_b200.binding` is the thin ctypes layer over it with the same names.
Importing this package does not load the library (so CPU-only tooling can import
`inputs`); any call into `binding` without the built library raises loudly.
"""
__all__ = ["binding", "inputs", "build"]
