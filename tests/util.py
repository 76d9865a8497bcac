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


class OnDevice:
    """numpy-style READ access to slices of a CUDA tensor.  The oracle only slices its big inputs (visibility
    rows of a subgrid, the master-grid patch under a subgrid); at the full sizes of BASELINE.json configs 3-5
    those arrays live on the device, and this hands the oracle the same numbers a slice at a time."""

    def __init__(self, t):
        self.t = t
        self.shape = tuple(t.shape)

    def __getitem__(self, idx):
        return self.t[idx].cpu().numpy()


def device_inner(a, b, chunk=1 << 24):
    """<a, b> = sum conj(a) b over two equally shaped complex64 CUDA tensors, accumulated in fp64 in chunks."""
    import torch
    fa, fb = a.reshape(-1), b.reshape(-1)
    acc = 0j
    for i in range(0, fa.numel(), chunk):
        x = fa[i:i + chunk].to(torch.complex128)
        y = fb[i:i + chunk].to(torch.complex128)
        acc += complex(torch.sum(torch.conj(x) * y).item())
    return acc
