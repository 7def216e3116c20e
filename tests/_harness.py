"""Helpers of the GPU parity tests: the call-sequence drivers live in the package (paper_2607_01065_b200/pipeline.py)."""
from paper_2607_01065_b200.pipeline import gpu_decode, gpu_gsrq, stats_np, to_device  # noqa: F401
