"""numpy front end of the fp64 CPU oracle (oracle/wstack_oracle.c) -- TEST INFRASTRUCTURE.

Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference leg may import
this module.  It imports nothing from paper_2301_06061_b200 and marshals numpy arrays only; all
arithmetic of the method is in the C file, each function there citing the PAPER.md passage it follows.
"""
from __future__ import annotations

import ctypes as C
import os
from dataclasses import dataclass
from typing import Optional, Sequence

import numpy as np

from . import build_oracle

_lib = None


class _Params(C.Structure):
    _fields_ = [("n_pix", C.c_int32), ("n_wplanes", C.c_int32), ("support", C.c_int32), ("tile", C.c_int32),
                ("sigma", C.c_double), ("cell_rad", C.c_double), ("w_min", C.c_double), ("w_max", C.c_double),
                ("kernel_type", C.c_int32), ("pad_", C.c_int32)]


KERNEL_GAUSSIAN = 0
KERNEL_KAISER_BESSEL = 1
NORM_SUMWT, NORM_N, NORM_TAPER = 1, 2, 4


@dataclass
class OracleParams:
    n_pix: int
    n_wplanes: int
    support: int
    cell_rad: float
    w_min: float
    w_max: float
    sigma: float = 1.0          # Gaussian: sigma in cells; Kaiser-Bessel: beta
    tile: int = 32
    kernel_type: int = 0

    def c(self) -> _Params:
        return _Params(self.n_pix, self.n_wplanes, self.support, self.tile, self.sigma, self.cell_rad,
                       self.w_min, self.w_max, self.kernel_type, 0)

    @property
    def n_bins(self) -> int:
        nt = self.n_pix // self.tile
        return self.n_wplanes * nt * nt


def lib():
    global _lib
    if _lib is None:
        _lib = C.CDLL(build_oracle.build())
        _lib.orc_bins.restype = C.c_int64
        _lib.orc_fft2.restype = C.c_int
        _lib.orc_num_threads.restype = C.c_int32
        for f in ("orc_i0", "orc_kernel1d", "orc_taper1d", "orc_sum_weights"):
            getattr(_lib, f).restype = C.c_double
    return _lib


def num_threads() -> int:
    return int(lib().orc_num_threads())


def _p(a, t):
    return a.ctypes.data_as(C.POINTER(t)) if a is not None else None


def _inputs(uvw, vis=None, wt=None, freq=None):
    uvw = np.ascontiguousarray(uvw, dtype=np.float32)
    assert uvw.ndim == 2 and uvw.shape[1] == 3
    if vis is not None:
        vis = np.ascontiguousarray(vis, dtype=np.complex64)
        wt = np.ascontiguousarray(wt, dtype=np.float32)
        assert vis.shape == wt.shape and vis.shape[0] == uvw.shape[0]
    fr = None if freq is None else np.ascontiguousarray(freq, dtype=np.float64)
    return uvw, vis, wt, fr


def channel_constants(prm: OracleParams, freq, n_chan):
    fr = None if freq is None else np.ascontiguousarray(freq, dtype=np.float64)
    su, sw, ow = np.empty(n_chan), np.empty(n_chan), C.c_double()
    lib().orc_channel_constants(C.byref(prm.c()), _p(fr, C.c_double), C.c_int32(n_chan),
                                _p(su, C.c_double), _p(sw, C.c_double), C.byref(ow))
    return su, sw, ow.value


def positions(prm: OracleParams, uvw, n_chan: int, freq=None):
    """O2-O4 for every visibility: dict of i0, j0, k (int32), fu, fv (float64), key (uint32)."""
    uvw, _, _, fr = _inputs(uvw, freq=freq)
    n = uvw.shape[0] * n_chan
    out = dict(i0=np.empty(n, np.int32), j0=np.empty(n, np.int32), k=np.empty(n, np.int32),
               fu=np.empty(n, np.float64), fv=np.empty(n, np.float64), key=np.empty(n, np.uint32))
    lib().orc_positions(C.byref(prm.c()), _p(uvw, C.c_float), C.c_int64(uvw.shape[0]), C.c_int32(n_chan),
                        _p(fr, C.c_double), _p(out["i0"], C.c_int32), _p(out["j0"], C.c_int32),
                        _p(out["k"], C.c_int32), _p(out["fu"], C.c_double), _p(out["fv"], C.c_double),
                        _p(out["key"], C.c_uint32))
    return out


def bins(prm: OracleParams, key: np.ndarray):
    """Stable counting sort by key -> (bin_start[n_bins+1] uint32, perm[n_kept] uint32, n_dropped)."""
    key = np.ascontiguousarray(key, dtype=np.uint32)
    bin_start = np.empty(prm.n_bins + 1, np.uint32)
    perm = np.empty(key.size, np.uint32)
    dropped = lib().orc_bins(_p(key, C.c_uint32), C.c_int64(key.size), C.c_int64(prm.n_bins),
                             _p(bin_start, C.c_uint32), _p(perm, C.c_uint32))
    return bin_start, perm[: key.size - dropped].copy(), int(dropped)


def grid(prm: OracleParams, uvw, vis, wt, freq=None, plane_lo: int = 0, plane_hi: Optional[int] = None,
         out: Optional[np.ndarray] = None) -> np.ndarray:
    """Eq. 3 onto planes [plane_lo, plane_hi): complex128 [n_planes, N, N], logical centred layout.
    If `out` is given the contributions are added to it (chunked gridding)."""
    uvw, vis, wt, fr = _inputs(uvw, vis, wt, freq)
    plane_hi = prm.n_wplanes if plane_hi is None else plane_hi
    N = prm.n_pix
    G = np.zeros((plane_hi - plane_lo, N, N), np.complex128) if out is None else out
    assert G.shape == (plane_hi - plane_lo, N, N) and G.dtype == np.complex128 and G.flags.c_contiguous
    lib().orc_grid(C.byref(prm.c()), _p(uvw, C.c_float), _p(vis.view(np.float32), C.c_float), _p(wt, C.c_float),
                   _p(fr, C.c_double), C.c_int64(uvw.shape[0]), C.c_int32(vis.shape[1]),
                   C.c_int32(plane_lo), C.c_int32(plane_hi), _p(G.view(np.float64), C.c_double))
    return G


def i0(x: float) -> float:
    return float(lib().orc_i0(C.c_double(x)))


def kernel1d(prm: OracleParams, x: float) -> float:
    """The 1-D convolution function g(x), x in cells (O5)."""
    return float(lib().orc_kernel1d(C.byref(prm.c()), C.c_double(x)))


def taper1d(prm: OracleParams, xi: float) -> float:
    """Continuous Fourier transform of g at xi cycles per cell."""
    return float(lib().orc_taper1d(C.byref(prm.c()), C.c_double(xi)))


def sum_weights(prm: OracleParams, uvw, wt, freq=None) -> float:
    uvw, _, _, fr = _inputs(uvw, freq=freq)
    wt = np.ascontiguousarray(wt, dtype=np.float32)
    return float(lib().orc_sum_weights(C.byref(prm.c()), _p(uvw, C.c_float), _p(wt, C.c_float), _p(fr, C.c_double),
                                       C.c_int64(uvw.shape[0]), C.c_int32(wt.shape[1])))


def dirty(prm: OracleParams, D: np.ndarray, flags: int = 0, sum_wt: float = 1.0) -> np.ndarray:
    """a5: Re D times the normalisation factors `flags` selects (NORM_SUMWT | NORM_N | NORM_TAPER)."""
    D = np.ascontiguousarray(D, dtype=np.complex128)
    out = np.empty(D.shape, np.float64)
    lib().orc_dirty(C.byref(prm.c()), _p(D.view(np.float64), C.c_double), C.c_uint32(flags), C.c_double(sum_wt),
                    _p(out, C.c_double))
    return out


def dft2_naive(plane: np.ndarray) -> np.ndarray:
    plane = np.ascontiguousarray(plane, dtype=np.complex128)
    N = plane.shape[0]
    assert plane.shape == (N, N)
    out = np.empty_like(plane)
    lib().orc_dft2_naive(C.c_int32(N), _p(plane.view(np.float64), C.c_double), _p(out.view(np.float64), C.c_double))
    return out


def fft2(plane: np.ndarray, inplace: bool = False) -> np.ndarray:
    x = plane if inplace else np.array(plane, dtype=np.complex128, order="C")
    assert x.dtype == np.complex128 and x.flags.c_contiguous and x.shape[0] == x.shape[1]
    rc = lib().orc_fft2(C.c_int32(x.shape[0]), _p(x.view(np.float64), C.c_double))
    if rc != 0:
        raise ValueError("oracle FFT needs a power-of-two size; use dft2_naive")
    return x


def transform(plane: np.ndarray, naive_max: int = 512) -> np.ndarray:
    """O7 for one plane: naive DFT for N <= naive_max, the oracle's FFT above."""
    return dft2_naive(plane) if plane.shape[0] <= naive_max else fft2(plane)


def wcorrect(prm: OracleParams, planes: np.ndarray, plane_lo: int = 0, out: Optional[np.ndarray] = None) -> np.ndarray:
    """Eq. 2: adds sum_k e^{2 pi i w_k (n-1)} P_k over the given planes to `out` (complex128 [N, N])."""
    planes = np.ascontiguousarray(planes, dtype=np.complex128)
    N = prm.n_pix
    D = np.zeros((N, N), np.complex128) if out is None else out
    lib().orc_wcorrect(C.byref(prm.c()), _p(planes.view(np.float64), C.c_double), C.c_int32(plane_lo),
                       C.c_int32(plane_lo + planes.shape[0]), _p(D.view(np.float64), C.c_double))
    return D


def transform_fwd(plane: np.ndarray, naive_max: int = 512) -> np.ndarray:
    """Forward un-normalised centred DFT (sign -): the conjugate of the inverse one of the conjugate."""
    return np.conj(transform(np.conj(np.asarray(plane, dtype=np.complex128)), naive_max))


def wscreen_fwd(prm: OracleParams, model: np.ndarray, k: int) -> np.ndarray:
    """Degridding step 1: model image times exp(-2 pi i w_k (n - 1))."""
    model = np.ascontiguousarray(model, dtype=np.complex128)
    out = np.empty_like(model)
    lib().orc_wscreen_fwd(C.byref(prm.c()), _p(model.view(np.float64), C.c_double), C.c_int32(k),
                          _p(out.view(np.float64), C.c_double))
    return out


def degrid(prm: OracleParams, uvw, n_chan: int, freq, planes: np.ndarray, plane_lo: int = 0,
           out: Optional[np.ndarray] = None) -> np.ndarray:
    """Degridding step 3 for the visibilities of planes [plane_lo, plane_lo + len(planes)): complex128 [n_rows, n_chan]."""
    uvw, _, _, fr = _inputs(uvw, freq=freq)
    planes = np.ascontiguousarray(planes, dtype=np.complex128)
    V = np.zeros((uvw.shape[0], n_chan), np.complex128) if out is None else out
    lib().orc_degrid(C.byref(prm.c()), _p(uvw, C.c_float), _p(fr, C.c_double), C.c_int64(uvw.shape[0]), C.c_int32(n_chan),
                     C.c_int32(plane_lo), C.c_int32(plane_lo + planes.shape[0]), _p(planes.view(np.float64), C.c_double),
                     _p(V.view(np.float64), C.c_double))
    return V


def predict(prm: OracleParams, model: np.ndarray, uvw, n_chan: int, freq=None, return_planes: bool = False,
            naive_max: int = 512):
    """The degridding chain, plane-streamed: w-screen -> forward transform -> gather.  complex128 [n_rows, n_chan]."""
    V = np.zeros((np.asarray(uvw).shape[0], n_chan), np.complex128)
    stack = [] if return_planes else None
    for k in range(prm.n_wplanes):
        H = transform_fwd(wscreen_fwd(prm, model, k), naive_max)
        if return_planes:
            stack.append(H)
        degrid(prm, uvw, n_chan, freq, H[None], k, V)
    return (V, np.stack(stack)) if return_planes else V


def predict_samples(prm: OracleParams, uvw, n_chan: int, freq, src_q, src_p, src_val, samples) -> np.ndarray:
    """The degridding chain at the visibilities `samples` (flat indices row * n_chan + c) for a sparse model image
    (pixels (src_q, src_p) with complex values src_val), visibility-outermost; complex128 [n_samples]."""
    uvw, _, _, fr = _inputs(uvw, freq=freq)
    sq = np.ascontiguousarray(src_q, dtype=np.int32)
    sp = np.ascontiguousarray(src_p, dtype=np.int32)
    sv = np.ascontiguousarray(src_val, dtype=np.complex128)
    samp = np.ascontiguousarray(samples, dtype=np.int64)
    out = np.empty(samp.size, np.complex128)
    lib().orc_predict_samples(C.byref(prm.c()), _p(uvw, C.c_float), _p(fr, C.c_double), C.c_int32(n_chan),
                              C.c_int32(sq.size), _p(sq, C.c_int32), _p(sp, C.c_int32), _p(sv.view(np.float64), C.c_double),
                              C.c_int64(samp.size), _p(samp, C.c_int64), _p(out.view(np.float64), C.c_double))
    return out


def image_samples(prm: OracleParams, uvw, vis, wt, freq, q: Sequence[int], p: Sequence[int]) -> np.ndarray:
    """The whole chain at pixels (q[s], p[s]), visibility-outermost; complex128 [n_samp]."""
    uvw, vis, wt, fr = _inputs(uvw, vis, wt, freq)
    q = np.ascontiguousarray(q, dtype=np.int32)
    p_ = np.ascontiguousarray(p, dtype=np.int32)
    out = np.empty(q.size, np.complex128)
    lib().orc_image_samples(C.byref(prm.c()), _p(uvw, C.c_float), _p(vis.view(np.float32), C.c_float),
                            _p(wt, C.c_float), _p(fr, C.c_double), C.c_int64(uvw.shape[0]), C.c_int32(vis.shape[1]),
                            C.c_int32(q.size), _p(q, C.c_int32), _p(p_, C.c_int32), _p(out.view(np.float64), C.c_double))
    return out


def dirty_image(prm: OracleParams, uvw, vis, wt, freq=None, return_grid: bool = False, naive_max: int = 512):
    """The full chain, plane-streamed: grid -> per-plane transform -> w-correction.
    Returns the complex image D (dirty = D.real), and the mesh stack if asked."""
    D = np.zeros((prm.n_pix, prm.n_pix), np.complex128)
    stack = [] if return_grid else None
    for k in range(prm.n_wplanes):
        G = grid(prm, uvw, vis, wt, freq, k, k + 1)
        if return_grid:
            stack.append(G[0].copy())
        wcorrect(prm, transform(G[0], naive_max)[None], k, D)
    return (D, np.stack(stack)) if return_grid else D
