"""paper_2606_21868_b200 -- B200-native (sm_100a) hot path of WiSP (arxiv/paper_2606_21868).

The product is `libwisp.so` (C ABI, `include/wisp.h`; CUDA sources in `csrc/`).  This package is the thin
Python binding: argument marshalling only -- every step of the path runs in the library's kernels.
There is no CPU fallback: loading fails loudly if the library has not been built, and `wisp_create`
fails with WISP_ECUDA without a CUDA device.
"""
from .binding import (  # noqa: F401
    WISP_BF16, WISP_F32, WISP_FP8_E4M3, WISP_FETCH_FUSED, WISP_FETCH_MEMCPY, WISP_FETCH_STATIC, WISP_FETCH_ZEROCOPY, WISP_LFU, WISP_LRU, WISP_WAVES_ASCENDING, WISP_WAVES_HITS_FIRST, WispConfig, WispError,
    WispLayerStats, WispMvwsaIn, WispStats, WispTraceEvent, Wisp, lib, lib_path, route_noalloc, STATUS_NAMES, KERNEL_CLASSES,
)
