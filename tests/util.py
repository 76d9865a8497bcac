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


def check_gridder_subgrids(idg, plan, par, obs, sub, vis, d_vis, d_at, d_tp, picks, window=64, tol=1e-5):
    """north_star's metric for the imaging direction, usable at any size: subgrid s after the gridder + A-term + taper
    (steps a1-a3, Eq. 10) and after the subgrid FFT (a4, :157) against the oracle's subgrid,
    max |gpu - oracle| / max |oracle| of THAT subgrid <= tol.  Each pick is computed inside a window of neighbouring
    subgrids through idg_grid_subgrids, i.e. with the plan's own kernel choice and launch configuration.
    `vis` is what the oracle slices (numpy array or OnDevice).  Returns (worst after a3, worst after a4, the
    gridder kernel mask of the windows)."""
    import torch
    L, n = par.subgrid_size, len(sub)
    worst = [0.0, 0.0]
    idg.kernel_config_mask("gridder", reset=True)
    for s in picks:
        first = min(max(0, s - window // 2), max(0, n - window))
        count = min(window, n - first)
        Sp, Shat = orc.grid_subgrid(par, sub[s], obs.uvw, obs.freqs, vis, obs.baselines, obs.aterms, obs.taper)
        out = torch.empty((count, 4, L, L), dtype=torch.complex64, device=d_vis.device)
        for k, (stage, want) in enumerate(((idg.STAGE_GRIDDER, Sp), (idg.STAGE_FFT, Shat))):
            out.fill_(float("nan"))
            idg.grid_subgrids(plan, first, count, d_vis, d_at, d_tp, out, stage=stage)
            got = np.moveaxis(out[s - first].cpu().numpy(), 0, 2)
            e = float(np.abs(got - want).max() / np.abs(want).max())
            assert e <= tol, (int(s), sub[s].tolist(), "gridder" if k == 0 else "fft", e)
            worst[k] = max(worst[k], e)
    return worst[0], worst[1], idg.kernel_config_mask("gridder", reset=True)
