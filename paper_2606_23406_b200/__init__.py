"""HyperQuant (arxiv/paper_2606_23406) inference hot path for NVIDIA B200 — thin Python binding of libhq.so.

All compute runs in the CUDA kernels behind the C ABI of include/hq.h; this package only marshals
arguments and lends torch's caching allocator and streams to the library.  There is no CPU path:
importing works anywhere (the library is dlopen'ed lazily), calling needs an sm_100 GPU.
"""
from .binding import (HQ_BF16, HQ_F32, Lattice, Context, Weight, KVCache, HQError, lib_path, load_library,
                      alpha, snr_for_bps, WeightHeader, EXPORTS, Layer, FOLD_NONE, FOLD_RMSNORM, FOLD_SILU_MUL, CAST_INT8, CAST_FP8_E4M3)

__all__ = ["HQ_BF16", "HQ_F32", "Lattice", "Context", "Weight", "KVCache", "HQError", "lib_path", "load_library",
           "alpha", "snr_for_bps", "WeightHeader", "EXPORTS", "Layer", "FOLD_NONE", "FOLD_RMSNORM", "FOLD_SILU_MUL", "CAST_INT8", "CAST_FP8_E4M3"]
