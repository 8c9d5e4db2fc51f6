"""B200-native w-stacking hot path (arxiv 2301.06061): thin Python binding over the C ABI of include/wstack.h.

PyTorch is used for device memory and streams only; every step runs in libwstack.so (hand-written CUDA for
sm_100a, cuFFT for the per-plane FFT).  There is no CPU fallback: importing `wstack` fails if the library
cannot be built or loaded.
"""
from .wstack import (WS_GRID_ACCUMULATE, WS_GRID_OVERWRITE, WS_FLAG_LIBRARY_FFT, WS_FLAG_NO_TRANSPOSE, WS_GRID_SPARSE, WS_GRID_SPARSE_ADD, WS_FFT_USE_OCCUPANCY, WS_VERSION, WS_FLAG_TRACK_SUMWT, WS_FLAG_PRESUM_CHANNELS, WS_FLAG_MESH_F64, WS_KERNEL_GAUSSIAN, WS_KERNEL_KAISER_BESSEL, WS_NORM_SUMWT, WS_NORM_N, WS_NORM_TAPER, Plan, WStackError, lib, library_path, static_scratch_bytes,  # noqa: F401
                     EXPORTED_SYMBOLS)
