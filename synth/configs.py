"""The five BASELINE.json workloads as generator recipes.

The paper's LOFAR HBA measurement sets (Table 2 :282-300) are not
available; these recipes stand in for them and keep their structure: snapshots
recorded one after the other with every baseline per snapshot (time-major rows,
PAPER.md:98), a core-dense station layout (:108), an hours-long track, and a
120-180 MHz band.
"""
from __future__ import annotations

from dataclasses import dataclass, field, replace
from typing import Optional, Tuple


@dataclass(frozen=True)
class ObsConfig:
    name: str
    seed: int
    # array
    layout: str                 # "disk" | "lofar_like" | "log_spiral"
    n_ant: int
    # track
    n_times: int
    hours: float
    dec_deg: float
    lat_deg: float = 53.0
    # band: Hz. narrow_band=True -> uvw handed over in wavelengths, freq=None
    freqs_hz: Tuple[float, ...] = (150e6,)
    narrow_band: bool = True
    n_shared_chan: int = 1      # narrow-band only: visibilities (channels x polarisations) per row sharing its uvw
    # sky model
    n_src: int = 5
    src_field: float = 0.1      # side of the square the sources fall in (rad); <0: fraction of FoV
    flux_law: str = "uniform"   # "uniform" U[0.1,1] | "powerlaw" pdf ~ F^-1.5 on [0.01,10]
    noise_sigma: float = 0.01
    weights: str = "unit"       # "unit" | "uniform" U[0.5,1.5]
    diffuse_rms: float = 0.0    # Large/Extreme: Gaussian random field term (Jy rms)
    # imaging parameters
    n_pix: int = 256
    n_wplanes: int = 4
    support: int = 7
    sigma_cells: float = 1.0
    # Extreme: rescale the layout so max(|u|,|v|) at the top frequency equals this (wavelengths)
    umax_lambda: Optional[float] = None
    cell_rad: Optional[float] = None   # None -> 1/(2 U)
    n_chunks: int = 1           # row chunks fed through repeated grid calls

    @property
    def n_baselines(self) -> int:
        return self.n_ant * (self.n_ant - 1) // 2

    @property
    def n_rows(self) -> int:
        return self.n_baselines * self.n_times

    @property
    def n_chan(self) -> int:
        return self.n_shared_chan if self.narrow_band else len(self.freqs_hz)

    @property
    def n_vis(self) -> int:
        return self.n_rows * self.n_chan

    def scaled(self, **kw) -> "ObsConfig":
        """A reduced copy (same recipe, smaller counts) for quick tests."""
        return replace(self, **kw)


def _band(lo_mhz: float, hi_mhz: float, n: int) -> Tuple[float, ...]:
    if n == 1:
        return (0.5 * (lo_mhz + hi_mhz) * 1e6,)
    step = (hi_mhz - lo_mhz) / (n - 1)
    return tuple((lo_mhz + i * step) * 1e6 for i in range(n))


CONFIGS = {
    # 24*23/2 = 276 baselines x 200 samples = 55,200 visibilities
    "tiny": ObsConfig(
        name="tiny", seed=1001, layout="disk", n_ant=24, n_times=200, hours=6.0, dec_deg=45.0,
        freqs_hz=(150e6,), narrow_band=True, n_src=5, src_field=0.1, flux_law="uniform",
        noise_sigma=0.01, weights="unit", n_pix=256, n_wplanes=4, support=7),
    # 1891 x 600 = 1,134,600
    "small": ObsConfig(
        name="small", seed=1002, layout="lofar_like", n_ant=62, n_times=600, hours=8.0, dec_deg=27.5,
        freqs_hz=(150e6,), narrow_band=True, n_src=50, src_field=0.2, flux_law="powerlaw",
        noise_sigma=0.05, weights="uniform", n_pix=2048, n_wplanes=16, support=7),
    # 1891 x 1800 x 4 = 13,615,200
    "medium": ObsConfig(
        name="medium", seed=1003, layout="lofar_like", n_ant=62, n_times=1800, hours=8.0, dec_deg=27.5,
        freqs_hz=_band(120, 180, 4), narrow_band=False, n_src=500, src_field=0.4, flux_law="powerlaw",
        noise_sigma=0.05, weights="uniform", n_pix=4096, n_wplanes=32, support=7),
    # 2016 x 6200 x 8 = 99,993,600
    "large": ObsConfig(
        name="large", seed=1004, layout="log_spiral", n_ant=64, n_times=6200, hours=8.0, dec_deg=27.5,
        freqs_hz=_band(120, 180, 8), narrow_band=False, n_src=2000, src_field=-0.8, flux_law="powerlaw",
        noise_sigma=0.05, weights="uniform", diffuse_rms=0.1, n_pix=8192, n_wplanes=64, support=7),
    # 2016 x 6200 x 32 = 399,974,400, eight row chunks of 775 snapshots
    "extreme": ObsConfig(
        name="extreme", seed=1005, layout="log_spiral", n_ant=64, n_times=6200, hours=8.0, dec_deg=27.5,
        freqs_hz=_band(120, 180, 32), narrow_band=False, n_src=2000, src_field=-0.8, flux_law="powerlaw",
        noise_sigma=0.05, weights="uniform", diffuse_rms=0.1, n_pix=16384, n_wplanes=32, support=9,
        umax_lambda=8100.0, cell_rad=1.0 / 16384, n_chunks=8),
    # the shape of the paper's own "Medium" test (Table 3: 0.54e9 visibilities, mesh
    # 4096 x 4096 x 16) in its narrow-band mode (:207, one uvw per measurement shared by all frequencies and
    # polarisations): 1891 baselines x 7200 samples = 13,615,200 rows x 40 (20 channels x 2 polarisations) = 544,608,000
    "paper_medium": ObsConfig(
        name="paper_medium", seed=1006, layout="lofar_like", n_ant=62, n_times=7200, hours=8.0, dec_deg=27.5,
        freqs_hz=(150e6,), narrow_band=True, n_shared_chan=40, n_src=500, src_field=0.2, flux_law="powerlaw",
        noise_sigma=0.05, weights="uniform", n_pix=4096, n_wplanes=16, support=7),
}


def get_config(name: str) -> ObsConfig:
    return CONFIGS[name.lower()]
