"""Seeded synthetic interferometer inputs.

This package only *produces inputs* (uvw, visibilities, weights, frequencies and
the scalar imaging parameters derived from them).  It holds none of the
w-stacking arithmetic (no gridding, no FFT, no w-correction) and is the one
module both the oracle tests and the CUDA path may share.
"""
from .configs import CONFIGS, ObsConfig, get_config  # noqa: F401
from .interferometer import Dataset, make_dataset, make_random_dataset  # noqa: F401
