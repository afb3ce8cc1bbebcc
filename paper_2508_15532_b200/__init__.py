"""B200-native radiation hot path of arxiv 2508.15532 (cuHARM radiation module).

The product is the C-ABI library `librt_b200.so` (include/rt.h, sources in csrc/); `rt.py` is its thin binding.
Build: `python -m paper_2508_15532_b200.build`.  There is no CPU fallback.
"""
__all__ = ["rt", "build"]
