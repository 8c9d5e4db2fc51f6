"""ctypes binding of libwstack.so -- argument marshalling only (same names as include/wstack.h)."""
from __future__ import annotations

import ctypes as C
import os
from typing import Optional, Sequence

import numpy as np
import torch

from . import build as _build

WS_VERSION = 200            # include/wstack.h
WS_GRID_ACCUMULATE = 0
WS_GRID_OVERWRITE = 1
WS_FLAG_LIBRARY_FFT = 1
WS_FLAG_NO_TRANSPOSE = 2
WS_GRID_SPARSE = 2
WS_GRID_SPARSE_ADD = 3
WS_FFT_USE_OCCUPANCY = 1
WS_FLAG_TRACK_SUMWT = 4
WS_FLAG_PRESUM_CHANNELS = 8
WS_FLAG_MESH_F64 = 16
WS_KERNEL_GAUSSIAN = 0
WS_KERNEL_KAISER_BESSEL = 1
WS_NORM_SUMWT, WS_NORM_N, WS_NORM_TAPER = 1, 2, 4

EXPORTED_SYMBOLS = [
    "ws_version", "ws_strerror", "ws_last_error", "ws_plan_create", "ws_plan_destroy", "ws_plan_set_snapshot_rows", "ws_plan_set_plane_range", "ws_grid_bytes",
    "ws_image_bytes", "ws_dirty_bytes", "ws_workspace_bytes", "ws_workspace_bytes_for", "ws_fft_workspace_bytes",
    "ws_plan_tile", "ws_plan_n_bins", "ws_grid_zero", "ws_grid_visibilities", "ws_bin_visibilities", "ws_grid_binned", "ws_fft_planes",
    "ws_wcorrect_accumulate", "ws_fft_wcorrect", "ws_fft_columns", "ws_fft_rows_wcorrect", "ws_plan_fft_is_own", "ws_get_occupancy", "ws_dirty_image", "ws_get_sum_weights", "ws_predict_planes", "ws_degrid_visibilities", "ws_predict_visibilities", "ws_dev_inputs_bytes", "ws_plan_set_e2e_chunk_bytes", "ws_image_from_host", "ws_get_bins", "ws_async_status",
    "ws_launch_count", "ws_measure_fp32_tflops", "ws_grid_visibilities_static", "ws_static_scratch_bytes",
]


class WStackError(RuntimeError):
    def __init__(self, code: int, msg: str):
        super().__init__(f"libwstack error {code}: {msg}")
        self.code = code


class _Params(C.Structure):
    _fields_ = [("n_pix", C.c_int32), ("n_wplanes", C.c_int32), ("support", C.c_int32), ("kernel_type", C.c_int32),
                ("kernel_param", C.c_double), ("cell_rad", C.c_double), ("w_min", C.c_double), ("w_max", C.c_double),
                ("tile", C.c_int32), ("device", C.c_int32), ("flags", C.c_uint32)]


_lib = None


def library_path() -> str:
    return _build.LIB


def lib():
    """Loads (building if needed) libwstack.so.  Raises if that is impossible: there is no fallback path."""
    global _lib
    if _lib is not None:
        return _lib
    path = _build.build()
    L = C.CDLL(path)
    vp, i32, i64, u32, sz = C.c_void_p, C.c_int32, C.c_int64, C.c_uint32, C.c_size_t
    sig = {
        "ws_version": (C.c_int, []),
        "ws_strerror": (C.c_char_p, [C.c_int]),
        "ws_last_error": (C.c_char_p, [vp]),
        "ws_plan_create": (C.c_int, [C.POINTER(_Params), C.POINTER(vp)]),
        "ws_plan_destroy": (C.c_int, [vp]),
        "ws_plan_set_snapshot_rows": (C.c_int, [vp, i64]),
        "ws_plan_set_plane_range": (C.c_int, [vp, i32, i32]),
        "ws_grid_bytes": (sz, [vp]), "ws_image_bytes": (sz, [vp]), "ws_dirty_bytes": (sz, [vp]),
        "ws_workspace_bytes": (sz, [vp, i64]),
        "ws_workspace_bytes_for": (sz, [vp, i64, C.c_double]),
        "ws_fft_workspace_bytes": (sz, [vp]),
        "ws_plan_tile": (C.c_int, [vp]), "ws_plan_n_bins": (i64, [vp]),
        "ws_grid_zero": (C.c_int, [vp, vp, vp]),
        "ws_grid_visibilities": (C.c_int, [vp, vp, vp, vp, C.POINTER(C.c_double), i64, i32, vp, i32, vp, sz, vp]),
        "ws_bin_visibilities": (C.c_int, [vp, vp, vp, vp, C.POINTER(C.c_double), i64, i32, vp, sz, vp]),
        "ws_grid_visibilities_static": (C.c_int, [vp, vp, vp, vp, C.POINTER(C.c_double), i64, i32, vp, i32, vp]),
        "ws_static_scratch_bytes": (sz, []),
        "ws_grid_binned": (C.c_int, [vp, vp, i32, vp, sz, vp]),
        "ws_fft_planes": (C.c_int, [vp, vp, vp, sz, vp]),
        "ws_wcorrect_accumulate": (C.c_int, [vp, vp, vp, i32, vp, vp]),
        "ws_fft_wcorrect": (C.c_int, [vp, vp, vp, i32, vp, u32, vp, sz, vp]),
        "ws_fft_columns": (C.c_int, [vp, vp, u32, vp]),
        "ws_fft_rows_wcorrect": (C.c_int, [vp, vp, vp, i32, vp, u32, vp]),
        "ws_plan_fft_is_own": (C.c_int, [vp]),
        "ws_get_occupancy": (C.c_int, [vp] + [C.POINTER(C.c_double)] * 4 + [C.POINTER(i32), vp]),
        "ws_dirty_image": (C.c_int, [vp, vp, vp, u32, vp]),
        "ws_get_sum_weights": (C.c_int, [vp, C.POINTER(C.c_double), vp]),
        "ws_predict_planes": (C.c_int, [vp, vp, vp, vp, sz, vp]),
        "ws_degrid_visibilities": (C.c_int, [vp, vp, C.POINTER(C.c_double), i64, i32, vp, vp, C.c_float, i32, vp, sz, vp]),
        "ws_predict_visibilities": (C.c_int, [vp, vp, vp, C.POINTER(C.c_double), i64, i32, vp, vp, C.c_float, i32, vp, sz, vp]),
        "ws_dev_inputs_bytes": (sz, [i64, i32]),
        "ws_plan_set_e2e_chunk_bytes": (C.c_int, [vp, sz]),
        "ws_image_from_host": (C.c_int, [vp, vp, vp, vp, C.POINTER(C.c_double), i64, i32, vp, sz, vp, vp, vp, vp, vp, sz, vp]),
        "ws_get_bins": (C.c_int, [vp, C.POINTER(vp), C.POINTER(vp), C.POINTER(vp), C.POINTER(vp), C.POINTER(i64),
                                  C.POINTER(i64), C.POINTER(i64), C.POINTER(i64), vp]),
        "ws_async_status": (C.c_int, [vp, vp]),
        "ws_launch_count": (i64, [vp]),
        "ws_measure_fp32_tflops": (C.c_int, [vp, C.POINTER(C.c_double), vp]),
    }
    for name, (res, args) in sig.items():
        fn = getattr(L, name)
        fn.restype, fn.argtypes = res, args
    if L.ws_version() != WS_VERSION:
        raise RuntimeError(f"libwstack.so is version {L.ws_version()}, the binding expects {WS_VERSION}: rebuild "
                           "(python -m paper_2301_06061_b200.build --force)")
    _lib = L
    return L


def static_scratch_bytes() -> int:
    """Size of the static device array behind Plan.grid_visibilities_static (WS_STATIC_SCRATCH_BYTES of the loaded library)."""
    return int(lib().ws_static_scratch_bytes())


def _stream(stream) -> int:
    s = torch.cuda.current_stream() if stream is None else stream
    return int(s.cuda_stream)


def _dev(t: torch.Tensor, dtype, name: str) -> int:
    if not (t.is_cuda and t.is_contiguous() and t.dtype == dtype):
        raise ValueError(f"{name}: expected a contiguous CUDA tensor of {dtype}")
    return t.data_ptr()


def _freq(freq_hz: Optional[Sequence[float]], n_chan: int):
    if freq_hz is None:
        return None, None
    arr = (C.c_double * n_chan)(*[float(f) for f in freq_hz])
    return arr, C.cast(arr, C.POINTER(C.c_double))


class Plan:
    """An imaging plan (ws_plan).  All buffers are torch CUDA tensors owned by the caller."""

    def __init__(self, n_pix: int, n_wplanes: int, support: int, cell_rad: float, w_min: float, w_max: float,
                 sigma: float = 1.0, tile: int = 0, device: int = 0, flags: int = 0,
                 kernel_type: int = WS_KERNEL_GAUSSIAN, kernel_param: Optional[float] = None):
        """kernel_param: Gaussian sigma in cells / Kaiser-Bessel beta; `sigma` is the older name of the same field."""
        self._h = C.c_void_p()
        prm = _Params(n_pix, n_wplanes, support, kernel_type, sigma if kernel_param is None else kernel_param,
                      cell_rad, w_min, w_max, tile, device, flags)
        rc = lib().ws_plan_create(C.byref(prm), C.byref(self._h))
        if rc != 0:
            self._h = C.c_void_p()
            raise WStackError(rc, lib().ws_strerror(rc).decode())
        self.n_pix, self.n_wplanes, self.support, self.device = n_pix, n_wplanes, support, device
        f64 = bool(flags & WS_FLAG_MESH_F64)        # fp64 mesh: complex128 grid / image, float64 dirty image
        self._c, self._r = (torch.complex128, torch.float64) if f64 else (torch.complex64, torch.float32)

    # -- plumbing ---------------------------------------------------------------------------------------
    def _check(self, rc: int):
        if rc != 0:
            raise WStackError(rc, lib().ws_last_error(self._h).decode() or lib().ws_strerror(rc).decode())

    def close(self):
        if getattr(self, "_h", None) and self._h.value:
            lib().ws_plan_destroy(self._h)
            self._h = C.c_void_p()

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    def set_snapshot_rows(self, rows_per_snapshot: int):
        """Performance hint: the input rows are time-major with this many rows (baselines) per snapshot."""
        self._check(lib().ws_plan_set_snapshot_rows(self._h, int(rows_per_snapshot)))

    def set_plane_range(self, plane_lo: int, plane_hi: int):
        """Keep only the visibilities of w-planes [plane_lo, plane_hi): this rank's share of a plane-sharded image."""
        self._check(lib().ws_plan_set_plane_range(self._h, int(plane_lo), int(plane_hi)))

    # -- sizes ------------------------------------------------------------------------------------------
    @property
    def tile(self) -> int:
        return lib().ws_plan_tile(self._h)

    @property
    def n_bins(self) -> int:
        return lib().ws_plan_n_bins(self._h)

    def grid_bytes(self) -> int:
        return lib().ws_grid_bytes(self._h)

    def image_bytes(self) -> int:
        return lib().ws_image_bytes(self._h)

    def workspace_bytes(self, max_vis: int, dup_factor: Optional[float] = None) -> int:
        if dup_factor is None:
            return lib().ws_workspace_bytes(self._h, max_vis)
        return lib().ws_workspace_bytes_for(self._h, max_vis, dup_factor)

    @property
    def fft_is_own(self) -> bool:
        return bool(lib().ws_plan_fft_is_own(self._h))

    def fft_workspace_bytes(self) -> int:
        return lib().ws_fft_workspace_bytes(self._h)

    def launch_count(self) -> int:
        return lib().ws_launch_count(self._h)

    # -- allocation helpers (torch owns the memory) ------------------------------------------------------
    def alloc_grid(self) -> torch.Tensor:
        return torch.empty((self.n_wplanes, self.n_pix, self.n_pix), dtype=self._c, device=f"cuda:{self.device}")

    def alloc_image(self) -> torch.Tensor:
        return torch.empty((self.n_pix, self.n_pix), dtype=self._c, device=f"cuda:{self.device}")

    def alloc_dirty(self) -> torch.Tensor:
        return torch.empty((self.n_pix, self.n_pix), dtype=self._r, device=f"cuda:{self.device}")

    def alloc_workspace(self, max_vis: int, dup_factor: Optional[float] = None) -> torch.Tensor:
        n = self.workspace_bytes(max_vis, dup_factor)
        return torch.empty((n + 255) // 256 * 256, dtype=torch.uint8, device=f"cuda:{self.device}")

    # -- the chain --------------------------------------------------------------------------------------
    def grid_zero(self, grid: torch.Tensor, stream=None):
        self._check(lib().ws_grid_zero(self._h, _dev(grid, self._c, "grid"), _stream(stream)))

    def grid_visibilities(self, uvw, vis, weights, freq_hz, grid, workspace, mode: int = WS_GRID_OVERWRITE, stream=None):
        n_rows = int(uvw.shape[0])
        n_chan = int(vis.shape[1]) if vis.dim() == 2 else 1
        keep, fp = _freq(freq_hz, n_chan)
        self._check(lib().ws_grid_visibilities(
            self._h, _dev(uvw, torch.float32, "uvw"), _dev(vis, torch.complex64, "vis"),
            _dev(weights, torch.float32, "weights"), fp, n_rows, n_chan, _dev(grid, self._c, "grid"), mode,
            _dev(workspace, torch.uint8, "workspace"), workspace.numel(), _stream(stream)))
        self._ws = workspace

    def grid_visibilities_static(self, uvw, vis, weights, freq_hz, grid, mode: int = WS_GRID_OVERWRITE, stream=None):
        """grid_visibilities with the workspace in the library's static device array (no allocation; see wstack.h for
        the size limit and the sharing rule)."""
        n_rows = int(uvw.shape[0])
        n_chan = int(vis.shape[1]) if vis.dim() == 2 else 1
        keep, fp = _freq(freq_hz, n_chan)
        self._check(lib().ws_grid_visibilities_static(
            self._h, _dev(uvw, torch.float32, "uvw"), _dev(vis, torch.complex64, "vis"),
            _dev(weights, torch.float32, "weights"), fp, n_rows, n_chan, _dev(grid, self._c, "grid"), mode, _stream(stream)))
        self._ws = None

    def bin_visibilities(self, uvw, vis, weights, freq_hz, workspace, stream=None):
        n_rows = int(uvw.shape[0])
        n_chan = int(vis.shape[1]) if vis.dim() == 2 else 1
        keep, fp = _freq(freq_hz, n_chan)
        self._check(lib().ws_bin_visibilities(
            self._h, _dev(uvw, torch.float32, "uvw"), _dev(vis, torch.complex64, "vis"),
            _dev(weights, torch.float32, "weights"), fp, n_rows, n_chan,
            _dev(workspace, torch.uint8, "workspace"), workspace.numel(), _stream(stream)))
        self._ws = workspace

    def grid_binned(self, grid, workspace, mode: int = WS_GRID_OVERWRITE, stream=None):
        self._check(lib().ws_grid_binned(self._h, _dev(grid, self._c, "grid"), mode,
                                         _dev(workspace, torch.uint8, "workspace"), workspace.numel(), _stream(stream)))

    def fft_planes(self, grid, workspace, stream=None):
        self._check(lib().ws_fft_planes(self._h, _dev(grid, self._c, "grid"),
                                        _dev(workspace, torch.uint8, "workspace"), workspace.numel(), _stream(stream)))

    def wcorrect_accumulate(self, planes, image, accumulate: bool = False, dirty=None, stream=None):
        d = None if dirty is None else _dev(dirty, self._r, "dirty")
        self._check(lib().ws_wcorrect_accumulate(self._h, _dev(planes, self._c, "planes"),
                                                 _dev(image, self._c, "image"), int(accumulate), d,
                                                 _stream(stream)))

    def fft_wcorrect(self, grid, image, workspace, accumulate: bool = False, dirty=None, fft_flags: int = 0, stream=None):
        """a3 + a4 in one call (the mesh is destroyed)."""
        d = None if dirty is None else _dev(dirty, self._r, "dirty")
        self._check(lib().ws_fft_wcorrect(self._h, _dev(grid, self._c, "grid"),
                                          _dev(image, self._c, "image"), int(accumulate), d, fft_flags,
                                          _dev(workspace, torch.uint8, "workspace"), workspace.numel(), _stream(stream)))

    def fft_columns(self, grid, fft_flags: int = 0, stream=None):
        self._check(lib().ws_fft_columns(self._h, _dev(grid, self._c, "grid"), fft_flags, _stream(stream)))

    def fft_rows_wcorrect(self, grid, image, accumulate: bool = False, dirty=None, fft_flags: int = 0, stream=None):
        d = None if dirty is None else _dev(dirty, self._r, "dirty")
        self._check(lib().ws_fft_rows_wcorrect(self._h, _dev(grid, self._c, "grid"),
                                               _dev(image, self._c, "image"), int(accumulate), d, fft_flags,
                                               _stream(stream)))

    def dirty_image(self, image, dirty, norm_flags: int = 0, stream=None):
        self._check(lib().ws_dirty_image(self._h, _dev(image, self._c, "image"),
                                         _dev(dirty, self._r, "dirty"), norm_flags, _stream(stream)))

    def predict_planes(self, model_image, planes, workspace, stream=None):
        """Degridding steps 1-2: planes[k] = forward FFT of model_image x exp(-2 pi i w_k (n - 1))."""
        self._check(lib().ws_predict_planes(self._h, _dev(model_image, torch.complex64, "model_image"),
                                            _dev(planes, self._c, "planes"),
                                            _dev(workspace, torch.uint8, "workspace"), workspace.numel(), _stream(stream)))

    def degrid_visibilities(self, uvw, freq_hz, n_chan: int, planes, vis_out, workspace, scale: float = 1.0,
                            accumulate: bool = False, stream=None):
        """Degridding step 3: vis_out (+)= scale x the footprint sums of `planes` at every visibility position."""
        n_rows = int(uvw.shape[0])
        keep, fp = _freq(freq_hz, n_chan)
        self._check(lib().ws_degrid_visibilities(
            self._h, _dev(uvw, torch.float32, "uvw"), fp, n_rows, n_chan, _dev(planes, self._c, "planes"),
            _dev(vis_out, torch.complex64, "vis_out"), float(scale), int(accumulate),
            _dev(workspace, torch.uint8, "workspace"), workspace.numel(), _stream(stream)))
        self._ws = workspace

    def predict_visibilities(self, model_image, uvw, freq_hz, n_chan: int, planes, vis_out, workspace, scale: float = 1.0,
                             accumulate: bool = False, stream=None):
        """Degridding in one call (`planes` is scratch): bins first, then only the wanted column bands are transformed."""
        n_rows = int(uvw.shape[0])
        keep, fp = _freq(freq_hz, n_chan)
        self._check(lib().ws_predict_visibilities(
            self._h, _dev(model_image, torch.complex64, "model_image"), _dev(uvw, torch.float32, "uvw"), fp, n_rows, n_chan,
            _dev(planes, self._c, "planes"), _dev(vis_out, torch.complex64, "vis_out"), float(scale), int(accumulate),
            _dev(workspace, torch.uint8, "workspace"), workspace.numel(), _stream(stream)))
        self._ws = workspace

    def sum_weights(self, stream=None) -> float:
        v = C.c_double()
        self._check(lib().ws_get_sum_weights(self._h, C.byref(v), _stream(stream)))
        return v.value

    def set_e2e_chunk_bytes(self, nbytes: int):
        """Input bytes per pipelined chunk of image_from_host (0: default)."""
        self._check(lib().ws_plan_set_e2e_chunk_bytes(self._h, int(nbytes)))

    @staticmethod
    def dev_inputs_bytes(n_rows: int, n_chan: int) -> int:
        return int(lib().ws_dev_inputs_bytes(n_rows, n_chan))

    def image_from_host(self, uvw_h, vis_h, weights_h, freq_hz, dev_inputs, grid, image, dirty_d, dirty_h, workspace,
                        stream=None):
        """The whole path from HOST tensors (pinned for asynchronous copies) to a host dirty image."""
        for t, dt, nm in ((uvw_h, torch.float32, "uvw_h"), (vis_h, torch.complex64, "vis_h"),
                          (weights_h, torch.float32, "weights_h"), (dirty_h, torch.float32, "dirty_h")):
            if t.is_cuda or not t.is_contiguous() or t.dtype != dt:
                raise ValueError(f"{nm}: expected a contiguous host tensor of {dt}")
        n_rows, n_chan = int(uvw_h.shape[0]), int(vis_h.shape[1])
        keep, fp = _freq(freq_hz, n_chan)
        self._check(lib().ws_image_from_host(
            self._h, uvw_h.data_ptr(), vis_h.data_ptr(), weights_h.data_ptr(), fp, n_rows, n_chan,
            _dev(dev_inputs, torch.uint8, "dev_inputs"), dev_inputs.numel(), _dev(grid, self._c, "grid"),
            _dev(image, self._c, "image"), _dev(dirty_d, torch.float32, "dirty_d"), dirty_h.data_ptr(),
            _dev(workspace, torch.uint8, "workspace"), workspace.numel(), _stream(stream)))

    def measure_fp32_tflops(self, stream=None) -> float:
        """Diagnostic: the fp32 FMA rate (TFLOP/s) of a register-only loop on this device."""
        v = C.c_double()
        self._check(lib().ws_measure_fp32_tflops(self._h, C.byref(v), _stream(stream)))
        return v.value

    def occupancy(self, stream=None) -> dict:
        """Fractions of the mesh marked non-empty by the gridding calls: tiles, classes, bands, planes."""
        v = [C.c_double() for _ in range(4)]
        tr = C.c_int32()
        self._check(lib().ws_get_occupancy(self._h, *[C.byref(x) for x in v], C.byref(tr), _stream(stream)))
        out = dict(zip(("tiles", "classes", "bands", "planes"), (x.value for x in v)))
        out["transposed"] = bool(tr.value)
        return out

    def async_status(self, stream=None):
        self._check(lib().ws_async_status(self._h, _stream(stream)))

    def get_bins(self, stream=None, fields=("keys", "sorted_keys", "perm", "bin_start")) -> dict:
        """Bins of the last grid call as numpy arrays (copied to the host; only `fields`): keys, sorted_keys, perm,
        bin_start; plus n_vis, n_bins, n_dropped, n_records."""
        names = ("keys", "sorted_keys", "perm", "bin_start")
        p = [C.c_void_p() for _ in range(4)]
        n = [C.c_int64() for _ in range(4)]
        ptr_args = [C.byref(x) if nm in fields else None for nm, x in zip(names, p)]
        self._check(lib().ws_get_bins(self._h, *ptr_args, *[C.byref(x) for x in n], _stream(stream)))
        n_vis, n_bins, n_dropped, n_records = (int(x.value) for x in n)
        ws = self._ws
        base = ws.data_ptr()

        def view(ptr, count):
            off = ptr.value - base
            return ws[off: off + 4 * count].view(torch.int32).cpu().numpy().view(np.uint32)

        n_kept = n_vis - n_dropped
        counts = dict(keys=n_vis, sorted_keys=n_kept, perm=n_kept, bin_start=n_bins + 1)
        out = dict(n_vis=n_vis, n_bins=n_bins, n_dropped=n_dropped, n_records=n_records)
        for nm, x in zip(names, p):
            if nm in fields:
                out[nm] = view(x, counts[nm])
        return out
