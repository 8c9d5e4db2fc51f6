"""Synthetic interferometer data: station layouts, (u,v,w) tracks, sky model, visibilities.

Recipe = SURVEY.md section 8(d).  All geometry is fp64 and cast to fp32 / complex64 at
the end; the scalar imaging parameters (cell size, w range) are then derived in fp64
from the *rounded* fp32 coordinates, so that every consumer sees the same numbers.

The visibilities follow PAPER.md:59 (Eq. 1, discretised over point sources, without
the 1/n factor):  V = sum_s F_s exp(-2 pi i (u l_s + v m_s + w (n_s - 1))) + noise.
Their values never influence timing, only error norms.

Heavy parts run through torch so that the large configs can be synthesised on the GPU
(`device="cuda"`); random numbers always come from numpy on the host, from four
independent streams spawned from the config seed in the order
layout, sources, noise, weights.
"""
from __future__ import annotations

import math
from dataclasses import dataclass
from typing import Optional, Tuple

import numpy as np
import torch

from .configs import ObsConfig

C_LIGHT = 299_792_458.0  # m/s
_NOISE_BLOCK_ROWS = 1 << 20  # fixed: part of the recipe (noise stream is drawn block by block)


@dataclass
class Dataset:
    """One workload: device-agnostic tensors + the scalar parameters of the imaging plan."""
    name: str
    uvw: torch.Tensor                 # [n_rows, 3] float32; metres if freqs_hz is not None else wavelengths
    vis: torch.Tensor                 # [n_rows, n_chan] complex64
    weights: torch.Tensor             # [n_rows, n_chan] float32
    freqs_hz: Optional[Tuple[float, ...]]   # None -> uvw already in wavelengths, shared by all channels
    n_pix: int
    n_wplanes: int
    support: int
    sigma_cells: float
    cell_rad: float
    w_min: float
    w_max: float
    n_chunks: int = 1
    # sky model, for tests that compare against the direct DFT of the model
    src_l: Optional[np.ndarray] = None
    src_m: Optional[np.ndarray] = None
    src_flux: Optional[np.ndarray] = None
    # rows per snapshot (= baselines) when the rows are time-major with every baseline per snapshot
    rows_per_snapshot: Optional[int] = None

    @property
    def n_rows(self) -> int:
        return int(self.uvw.shape[0])

    @property
    def n_chan(self) -> int:
        return int(self.vis.shape[1])

    @property
    def n_vis(self) -> int:
        return self.n_rows * self.n_chan

    def to(self, device) -> "Dataset":
        d = Dataset(**{**self.__dict__})
        d.uvw, d.vis, d.weights = self.uvw.to(device), self.vis.to(device), self.weights.to(device)
        return d

    def chan_scale(self) -> np.ndarray:
        """Per-channel factor turning the stored uvw into wavelengths (fp64)."""
        if self.freqs_hz is None:
            return np.ones(self.n_chan, dtype=np.float64)
        return np.asarray(self.freqs_hz, dtype=np.float64) / C_LIGHT

    def row_chunks(self):
        """Row ranges [lo, hi) of the n_chunks snapshot-aligned chunks (Extreme)."""
        edges = np.linspace(0, self.n_rows, self.n_chunks + 1).astype(np.int64)
        return [(int(edges[i]), int(edges[i + 1])) for i in range(self.n_chunks)]


# ----------------------------------------------------------------------------- layouts
def _layout_disk(rng, n_ant, diameter_m=1000.0):
    r = 0.5 * diameter_m * np.sqrt(rng.random(n_ant))
    az = 2.0 * np.pi * rng.random(n_ant)
    return r * np.sin(az), r * np.cos(az)


def _layout_lofar_like(rng, n_ant, r_lo=25.0, r_hi=1500.0, min_sep=25.0):
    e, n = [], []
    while len(e) < n_ant:
        r = math.exp(rng.uniform(math.log(r_lo), math.log(r_hi)))
        az = rng.uniform(0.0, 2.0 * np.pi)
        x, y = r * math.sin(az), r * math.cos(az)
        if all((x - a) ** 2 + (y - b) ** 2 >= min_sep ** 2 for a, b in zip(e, n)):
            e.append(x)
            n.append(y)
    return np.asarray(e), np.asarray(n)


def _layout_log_spiral(rng, n_ant, r_lo=100.0, r_hi=25000.0, n_arms=3, pitch=1.1, jitter=0.02):
    s = np.arange(n_ant)
    arm, idx = s % n_arms, s // n_arms
    frac = idx / max(1, (n_ant - 1) // n_arms)
    r = r_lo * (r_hi / r_lo) ** frac
    az = arm * (2.0 * np.pi / n_arms) + pitch * np.log(r / r_lo)
    r = r * (1.0 + jitter * rng.standard_normal(n_ant))
    az = az + jitter * rng.standard_normal(n_ant)
    return r * np.sin(az), r * np.cos(az)


_LAYOUTS = {"disk": _layout_disk, "lofar_like": _layout_lofar_like, "log_spiral": _layout_log_spiral}


def _baseline_vectors(east, north, lat_rad):
    """ENU (up = 0) -> equatorial baseline components (Lx, Ly, Lz), baselines a<b lexicographic."""
    x = -math.sin(lat_rad) * north
    y = east
    z = math.cos(lat_rad) * north
    ia, ib = np.triu_indices(len(east), k=1)
    return x[ib] - x[ia], y[ib] - y[ia], z[ib] - z[ia]


def _uvw_tracks(lx, ly, lz, n_times, hours, dec_rad):
    """Textbook (u,v,w)(H, dec) rotation; hour angle evenly sampled, centred on transit.
    Returns fp64 [n_times * n_bl, 3] in time-major order."""
    h = (np.arange(n_times) + 0.5 - 0.5 * n_times) / n_times * (hours * 15.0 * np.pi / 180.0)
    sh, ch = np.sin(h)[:, None], np.cos(h)[:, None]
    sd, cd = math.sin(dec_rad), math.cos(dec_rad)
    u = sh * lx + ch * ly
    v = -sd * ch * lx + sd * sh * ly + cd * lz
    w = cd * ch * lx - cd * sh * ly + sd * lz
    return np.stack([u.ravel(), v.ravel(), w.ravel()], axis=1)


# ----------------------------------------------------------------------------- sky model
def _draw_sources(rng, cfg: ObsConfig, fov_rad: float):
    side = cfg.src_field if cfg.src_field > 0 else -cfg.src_field * fov_rad
    l = rng.uniform(-0.5 * side, 0.5 * side, cfg.n_src)
    m = rng.uniform(-0.5 * side, 0.5 * side, cfg.n_src)
    if cfg.flux_law == "uniform":
        f = rng.uniform(0.1, 1.0, cfg.n_src)
    else:  # pdf ~ F^-1.5 on [0.01, 10]: inverse-cdf sampling
        a, lo, hi = -0.5, 0.01, 10.0
        q = rng.random(cfg.n_src)
        f = (lo ** a + q * (hi ** a - lo ** a)) ** (1.0 / a)
    return l, m, f


def _diffuse_lattice(rng, rms, n=1024, index=3.0):
    k = np.hypot(*np.meshgrid(np.arange(n) - n // 2, np.arange(n) - n // 2, indexing="ij"))
    k[k < 1.0] = 1.0
    amp = k ** (-0.5 * index)
    fld = (rng.standard_normal((n, n)) + 1j * rng.standard_normal((n, n))) * amp
    fld *= rms / math.sqrt(float(np.mean(np.abs(fld) ** 2)))
    return fld.astype(np.complex64)


# ----------------------------------------------------------------------------- main entry
def make_dataset(cfg: ObsConfig, device="cpu", with_noise=True) -> Dataset:
    """Build the dataset for one config.  `device` only selects where the visibility
    synthesis runs and where the returned tensors live."""
    dev = torch.device(device)
    ss = np.random.SeedSequence(cfg.seed)
    rng_layout, rng_src, rng_noise, rng_wt = (np.random.default_rng(s) for s in ss.spawn(4))

    east, north = _LAYOUTS[cfg.layout](rng_layout, cfg.n_ant)
    lx, ly, lz = _baseline_vectors(east, north, math.radians(cfg.lat_deg))
    uvw_m = _uvw_tracks(lx, ly, lz, cfg.n_times, cfg.hours, math.radians(cfg.dec_deg))  # metres, fp64

    scale = np.asarray(cfg.freqs_hz, dtype=np.float64) / C_LIGHT     # metres -> wavelengths per channel
    if cfg.umax_lambda is not None:   # Extreme: rescale the layout to a prescribed uv extent
        uvw_m *= cfg.umax_lambda / (np.abs(uvw_m[:, :2]).max() * scale.max())

    if cfg.narrow_band:
        uvw32 = (uvw_m * scale[0]).astype(np.float32)   # handed over in wavelengths
        freqs, ch_scale = None, np.ones(1)
    else:
        uvw32 = uvw_m.astype(np.float32)                # metres + per-channel f/c
        freqs, ch_scale = tuple(cfg.freqs_hz), scale
    del uvw_m

    # scalar plan parameters, fp64, from the rounded coordinates
    uvw64 = uvw32.astype(np.float64)
    umax = float(np.abs(uvw64[:, :2]).max() * ch_scale.max())
    cell = cfg.cell_rad if cfg.cell_rad is not None else 1.0 / (2.0 * umax)
    wl = np.multiply.outer(uvw64[:, 2], ch_scale)
    w_min, w_max = float(wl.min()), float(wl.max())
    del wl

    l, m, flux = _draw_sources(rng_src, cfg, cfg.n_pix * cell)
    nm1 = -(l * l + m * m) / (1.0 + np.sqrt(1.0 - l * l - m * m))
    lattice = _diffuse_lattice(rng_src, cfg.diffuse_rms) if cfg.diffuse_rms > 0 else None

    n_rows, n_chan = uvw32.shape[0], len(ch_scale)
    n_shared = cfg.n_shared_chan if cfg.narrow_band else 1
    vis = torch.empty((n_rows, n_chan * n_shared), dtype=torch.complex64, device=dev)
    lmn = torch.tensor(np.stack([l, m, nm1], axis=0), dtype=torch.float64, device=dev)     # [3, n_src]
    flx = torch.tensor(flux, dtype=torch.complex128, device=dev)
    sc = torch.tensor(ch_scale, dtype=torch.float64, device=dev)
    lat_t = torch.tensor(lattice, device=dev) if lattice is not None else None
    rows_per_block = max(1, (1 << 25) // max(1, n_chan * cfg.n_src))
    n_out = n_chan * n_shared
    uvw_t = torch.from_numpy(uvw32).to(dev)
    for lo in range(0, n_rows, rows_per_block):
        hi = min(n_rows, lo + rows_per_block)
        p = uvw_t[lo:hi].double()                                   # [r, 3]
        pl = (p[:, None, :] * sc[None, :, None]).reshape(-1, 3)     # [r*n_chan, 3] wavelengths
        ph = pl @ lmn                                               # turns
        ph -= torch.round(ph)
        v = torch.polar(torch.ones_like(ph), ph * (-2.0 * math.pi)) @ flx
        if lat_t is not None:
            nl = lat_t.shape[0]
            iu = torch.clamp(torch.round((pl[:, 0] / umax * 0.5 + 0.5) * (nl - 1)).long(), 0, nl - 1)
            iv = torch.clamp(torch.round((pl[:, 1] / umax * 0.5 + 0.5) * (nl - 1)).long(), 0, nl - 1)
            v = v + lat_t[iv, iu]
        if n_shared > 1:      # narrow band: every channel / polarisation of the row sees the same model visibility
            vis[lo:hi] = v.reshape(hi - lo, 1).to(torch.complex64).expand(hi - lo, n_shared)
        else:
            vis[lo:hi] = v.reshape(hi - lo, n_chan).to(torch.complex64)
    if with_noise and cfg.noise_sigma > 0:
        for lo in range(0, n_rows, _NOISE_BLOCK_ROWS):
            hi = min(n_rows, lo + _NOISE_BLOCK_ROWS)
            z = rng_noise.standard_normal((hi - lo, n_out, 2), dtype=np.float32) * np.float32(cfg.noise_sigma)
            vis[lo:hi] += torch.view_as_complex(torch.from_numpy(z)).to(dev)

    if cfg.weights == "unit":
        wt = torch.ones((n_rows, n_out), dtype=torch.float32, device=dev)
    else:
        wt = torch.empty((n_rows, n_out), dtype=torch.float32, device=dev)
        for lo in range(0, n_rows, _NOISE_BLOCK_ROWS):
            hi = min(n_rows, lo + _NOISE_BLOCK_ROWS)
            wt[lo:hi] = torch.from_numpy(
                (0.5 + rng_wt.random((hi - lo, n_out), dtype=np.float32)).astype(np.float32)).to(dev)

    return Dataset(name=cfg.name, uvw=uvw_t, vis=vis, weights=wt, freqs_hz=freqs,
                   n_pix=cfg.n_pix, n_wplanes=cfg.n_wplanes, support=cfg.support,
                   sigma_cells=cfg.sigma_cells, cell_rad=float(cell), w_min=w_min, w_max=w_max,
                   n_chunks=cfg.n_chunks, src_l=l, src_m=m, src_flux=flux, rows_per_snapshot=cfg.n_baselines)


def make_random_dataset(seed: int, n_rows: int, n_chan: int, n_pix: int, n_wplanes: int, support: int,
                        *, wavelengths: bool = True, fill: float = 0.9, w_span: float = 50.0,
                        cell_rad: float = 1e-3, sigma_cells: float = 1.0, unit_weights: bool = False) -> Dataset:
    """Unstructured random visibilities for edge-case tests: uv uniform in `fill` x the grid extent
    (fill > 1 puts some outside, exercising the drop rule), w uniform in +-w_span wavelengths."""
    rng = np.random.default_rng(seed)
    half_extent = 0.5 / cell_rad           # |u| at the grid edge, wavelengths
    if wavelengths:
        freqs, top = None, 1.0
    else:
        fr = np.linspace(120e6, 180e6, n_chan) if n_chan > 1 else np.array([150e6])
        freqs, top = tuple(float(f) for f in fr), float(fr.max()) / C_LIGHT
    uv = rng.uniform(-fill * half_extent, fill * half_extent, (n_rows, 2)) / top
    w = rng.uniform(-w_span, w_span, (n_rows, 1)) / top
    uvw32 = np.concatenate([uv, w], axis=1).astype(np.float32)
    vis = (rng.standard_normal((n_rows, n_chan)) + 1j * rng.standard_normal((n_rows, n_chan))).astype(np.complex64)
    wt = np.ones((n_rows, n_chan), np.float32) if unit_weights else \
        rng.uniform(0.5, 1.5, (n_rows, n_chan)).astype(np.float32)
    ch = np.ones(1) if freqs is None else np.asarray(freqs) / C_LIGHT
    wl = np.multiply.outer(uvw32[:, 2].astype(np.float64), ch) if n_rows else np.zeros((1, 1))
    w_min, w_max = float(wl.min()), float(wl.max())
    if not w_max > w_min:
        w_min, w_max = w_min - 1.0, w_min + 1.0
    return Dataset(name=f"random{seed}", uvw=torch.from_numpy(uvw32), vis=torch.from_numpy(vis),
                   weights=torch.from_numpy(wt), freqs_hz=freqs, n_pix=n_pix, n_wplanes=n_wplanes,
                   support=support, sigma_cells=sigma_cells, cell_rad=cell_rad, w_min=w_min, w_max=w_max)
