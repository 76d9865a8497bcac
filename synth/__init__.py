"""Seeded synthetic observations (inputs only) for the IDG hot path.

This module holds *no arithmetic of the method* (no planner, phasor sums, A-term
sandwich, FFT, adder or splitter).  It only manufactures inputs with the shapes, sizes and
value distributions of the five workloads in BASELINE.json:
station layouts, uvw tracks, channel frequencies, point-source visibilities, per-station
A-term Jones maps and the Kaiser-Bessel taper.  Both the fp64 oracle (`oracle/`) and the CUDA
path (`paper_2502_17789_b200/`) are fed from here; neither imports the other.

The paper's own data (an MWA snapshot, and a simulated 32-minute MWA set,
PAPER.md §6.2) are not available; these seeded generators stand in for them.
"""
from .configs import CONFIGS, Config, get_config, scaled  # noqa: F401
from .generate import (  # noqa: F401
    Observation,
    aterms,
    baselines,
    channel_freqs,
    hash_visibilities,
    hash_visibilities_torch,
    kaiser_bessel_1d,
    make_observation,
    point_sources,
    source_visibilities,
    source_visibilities_torch,
    station_layout,
    taper_full_1d,
    taper_subgrid,
    uvw_metres,
)
