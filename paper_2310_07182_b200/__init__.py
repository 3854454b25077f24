"""paper_2310_07182_b200 -- B200-native (sm_100a) hot path of "Generate Coherent Rays Directly" (arxiv 2310.07182).

The product is libcrt.so (C ABI in include/crt.h, CUDA kernels in csrc/); `api` is its thin ctypes binding.
There is no CPU fallback: the binding raises when the library or a CUDA device is missing.
"""
from .api import (  # noqa: F401
    Context, Bvh, CrtError, Frame, Order, Camera, SceneMats, make_frame, make_order, order_for_tile, make_camera, crt_layout, lib, hit_prims, path_flags,
    MODES, MODE_INDEPENDENT, MODE_MORTON_REORDER, MODE_DIRECT_REUSE, EXPORTS,
)
