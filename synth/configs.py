"""The five workload shapes of BASELINE.json `configs`.

Only shapes and seeds live here.  Cell sizes are chosen so that |uv|max*S + L/2 < Ng/2
(the configs fix only Ng); see DESIGN.md "Input recipe".
"""
from __future__ import annotations

import dataclasses
import math

ARCSEC = math.pi / 180.0 / 3600.0


@dataclasses.dataclass(frozen=True)
class Config:
    config_id: int
    name: str
    n_stations: int
    layout: str            # "disk" | "ska"
    disk_diameter_m: float
    n_times: int
    dt_s: float
    n_chan: int
    chan_width_hz: float
    freq_hz: float         # first channel if freq_is_start else band centre
    freq_is_start: bool
    n_sources: int
    source_kind: str       # "uniform_flux" | "powerlaw"
    subgrid_size: int      # L
    padding: int           # P (total, both sides)
    grid_size: int         # Ng
    cell_arcsec: float
    aterm_period: int
    aterm_kind: str        # "fourier" | "beam_screen" | "array_factor"
    screen_rms: float
    screen_smooth: bool
    w_step: float          # wavelengths; 0 => single layer
    ha_mid_deg: float
    comfort: float = 0.75

    @property
    def seed(self) -> int:
        return 1000 + self.config_id

    @property
    def n_baselines(self) -> int:
        return self.n_stations * (self.n_stations - 1) // 2

    @property
    def n_rows(self) -> int:
        return self.n_baselines * self.n_times

    @property
    def n_vis(self) -> int:
        return self.n_rows * self.n_chan

    @property
    def cell_size(self) -> float:
        return self.cell_arcsec * ARCSEC

    @property
    def image_size(self) -> float:       # S = Ng * cell  (direction cosines)
        return self.grid_size * self.cell_size

    @property
    def n_intervals(self) -> int:
        return -(-self.n_times // self.aterm_period)


CONFIGS = {
    1: Config(1, "tiny", 8, "disk", 1000.0, 16, 2.0, 4, 40e3, 150e6, True, 5, "uniform_flux",
              32, 8, 512, 60.0, 8, "fourier", 0.1, True, 0.0, 0.0),
    2: Config(2, "mwa1", 128, "disk", 1500.0, 56, 2.0, 32, 40e3, 154e6, False, 200, "powerlaw",
              64, 12, 4096, 30.0, 8, "beam_screen", 0.5, True, 0.0, 0.0),
    3: Config(3, "mwa_long", 128, "disk", 5000.0, 96, 2.0, 384, 40e3, 154e6, False, 200, "powerlaw",
              96, 18, 8000, 20.0, 4, "beam_screen", 2.0, False, 50.0, 5.0),
    4: Config(4, "ska_low", 512, "ska", 1000.0, 32, 1.0, 64, 5.4e3, 110e6, False, 1000, "powerlaw",
              64, 12, 16384, 4.0, 4, "array_factor", 0.3, False, 0.0, 0.0),
    # config 5 = degridding-only prediction at config-3 shapes (same observation, random model grid)
    5: Config(5, "predict_long", 128, "disk", 5000.0, 96, 2.0, 384, 40e3, 154e6, False, 200, "powerlaw",
              96, 18, 8000, 20.0, 4, "beam_screen", 2.0, False, 50.0, 5.0),
}


def get_config(config_id: int) -> Config:
    return CONFIGS[int(config_id)]


def scaled(cfg: Config, *, n_stations: int | None = None, n_times: int | None = None,
           n_chan: int | None = None, **over) -> Config:
    """A reduced copy of a config (same geometry recipe, fewer stations/times/channels).

    Used by the CPU tests so the fp64 oracle finishes in seconds while the subgrid size,
    padding, grid and cell -- hence tile counts and ragged tails -- stay those of the config.
    """
    kw = dict(over)
    if n_stations is not None:
        kw["n_stations"] = n_stations
    if n_times is not None:
        kw["n_times"] = n_times
    if n_chan is not None:
        kw["n_chan"] = n_chan
    return dataclasses.replace(cfg, **kw)
