"""Shared test helpers: config -> oracle parameters, small custom observations."""
from __future__ import annotations

import dataclasses

import numpy as np

import synth
from oracle import idg_oracle as orc


def oracle_params(cfg) -> orc.OracleParams:
    return orc.OracleParams(grid_size=cfg.grid_size, subgrid_size=cfg.subgrid_size, padding=cfg.padding,
                            cell_size=cfg.cell_size, w_step=cfg.w_step, n_times=cfg.n_times,
                            n_chan=cfg.n_chan, aterm_period=cfg.aterm_period, comfort=cfg.comfort)


def tiny_config(**over):
    """Config-1-like observation with L | Ng so the closure identities of P1/P2/P5 are exact."""
    base = synth.get_config(1)
    kw = dict(n_stations=6, n_times=8, n_chan=4, grid_size=256, cell_arcsec=120.0, aterm_period=4)
    kw.update(over)
    return dataclasses.replace(base, **kw)


def random_jones(rng, shape, scale=0.3):
    """I + scale * CN(0,1) Jones maps of the given leading shape (+ (2,2))."""
    z = (rng.standard_normal(shape + (2, 2)) + 1j * rng.standard_normal(shape + (2, 2))) / np.sqrt(2.0)
    return (np.eye(2)[(None,) * len(shape)] + scale * z).astype(np.complex64)


def inner(a, b):
    """<a, b> = sum conj(a) b over every complex entry."""
    return np.vdot(np.asarray(a).ravel(), np.asarray(b).ravel())
