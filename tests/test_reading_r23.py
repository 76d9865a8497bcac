"""DESIGN.md reading R23, backed by the oracle alone (no GPU, none of the CUDA path's code).

Config 5 predicts visibilities from a model image that was divided by the image-level taper T_full (Eq. 12,
PAPER.md:166, reading R4).  Towards the edge of the field 1 / T_full grows without bound (Kaiser-Bessel with
P = 18: 6e4 per axis at 0.8 x the half field, 3e9 in a corner), and the prediction of a subgrid (Eq. 13,
PAPER.md:171-174) then comes out of a cancellation: the inverse subgrid transform leaves a peak of height
flux / T_full and sidelobes of that peak all over the subgrid, the subgrid taper multiplies the peak back down to
~flux, and the direct sum has to cancel the sidelobes against each other.

This file shows, with the fp64 oracle and a library FFT, WHERE a single-precision chain loses the 1e-5 bar on such
a model, whichever kernels it is made of:
  * storing the image-domain subgrid as complex64 (one `astype` on the oracle's fp64 subgrid) costs nothing
    (< 1e-6): every sample keeps its own relative accuracy, the sidelobes near the centre included;
  * computing the inverse L x L transform in single precision (scipy's pocketfft on complex64, an implementation
    this repository shares nothing with) leaves an error relative to the PEAK on every sample, ~1e-7 x flux /
    T_full, which the taper does not scale down near the subgrid's centre: sources in the inner half of the field
    stay below 1e-5, sources at 0.65 x and 0.8 x the half field exceed it.
So the floor belongs to the fp32 inverse transform of the subgrid stack, a step the fp64 kernel variant does not
replace (PAPER.md:371 speaks of the two direct sums), and tests/test_gpu_fullsize.py places the R23 model's sources
in the inner half; the BASELINE.json-literal model (no 1 / T_full) is tested there without that restriction.
"""
import numpy as np
import pytest
import scipy.fft

import synth
from oracle import idg_oracle as orc
from tests.util import oracle_params


def _case():
    # config 5's subgrid geometry (L = 96, P = 18, same image extent S, same w-step) on a 10x coarser image raster
    # and a 450 m array, so that the oracle finishes in seconds
    cfg = synth.scaled(synth.get_config(5), n_stations=5, n_times=8, n_chan=64, grid_size=800, cell_arcsec=200.0,
                       disk_diameter_m=450.0)
    obs = synth.make_observation(cfg, vis=None)
    par = oracle_params(cfg)
    sub, _ = orc.plan(par, obs.uvw, obs.freqs, cfg.n_baselines)
    assert len(sub) >= 10
    return cfg, obs, par, sub


def _model_grid(cfg, par, sub, frac, rng, n_src=4):
    """Master grid (complex64, as the device path receives it) of n_src point sources in the corners of the square
    of half-width frac x the half field, each flux / T_full: the transform of a delta is written out per source."""
    Ng = cfg.grid_size
    wl_min, W = orc.layer_range(sub)
    t1 = synth.taper_full_1d(Ng, cfg.padding)
    j = np.arange(Ng) - Ng // 2
    G = np.zeros((W, 4, Ng, Ng), np.complex128)
    r = int(frac * Ng / 2)
    for k in range(n_src):
        jy, jx = Ng // 2 + r * rng.choice([-1, 1]) - k, Ng // 2 + r * rng.choice([-1, 1]) - 2 * k
        flux = 10.0 ** rng.uniform(-1, 1, 4) * np.exp(2j * np.pi * rng.random(4))
        amp = flux / (t1[jy] * t1[jx])
        l, m = (jx - Ng // 2) * par.image_size / Ng, (jy - Ng // 2) * par.image_size / Ng
        ey, ex = np.exp(-2j * np.pi * j * (jy - Ng // 2) / Ng), np.exp(-2j * np.pi * j * (jx - Ng // 2) / Ng)
        for layer in range(W):
            w0 = (wl_min + layer + 0.5) * par.w_step
            G[layer] += amp[:, None, None] * np.exp(-2j * np.pi * w0 * orc.nprime(l, m)) * np.outer(ey, ex)[None]
    return G.astype(np.complex64), wl_min


def _errors(frac, seed=0):
    cfg, obs, par, sub = _case()
    rng = np.random.default_rng(seed)
    G, wl_min = _model_grid(cfg, par, sub, frac, rng)
    L = cfg.subgrid_size
    occ = sub[:, 2] * sub[:, 4]
    picks = sorted(set(rng.choice(len(sub), 5, replace=False).tolist()) | {int(occ.argmax())})
    e_store = e_fft = 0.0
    for s in picks:
        patch = orc.splitter(G, sub[s], L, wl_min)
        S = orc.subgrid_ifft(patch)
        Mp, Mq = orc.subgrid_jones(par, sub[s], obs.baselines, obs.aterms, obs.uvw)

        def predict(Sx):
            return orc.degridder_subgrid(par, sub[s], obs.uvw, obs.freqs, orc.aterm_taper(Sx, Mp, Mq, obs.taper))

        ref = predict(S)
        scale = np.abs(ref).max()
        e_store = max(e_store, np.abs(predict(S.astype(np.complex64)) - ref).max() / scale)
        p32 = np.ascontiguousarray(patch.astype(np.complex64))
        S32 = scipy.fft.fftshift(scipy.fft.ifft2(scipy.fft.ifftshift(p32, axes=(0, 1)), axes=(0, 1)), axes=(0, 1))
        assert S32.dtype == np.complex64, "the library transform must run in single precision"
        assert np.abs(S32 - S).max() <= 1e-5 * np.abs(S).max(), "same centred transform, same 1 / L^2"
        e_fft = max(e_fft, np.abs(predict(S32) - ref).max() / scale)
    return e_store, e_fft


@pytest.mark.parametrize("frac,inside", [(0.4, True), (0.5, True), (0.65, False), (0.8, False)])
def test_r23_floor_is_the_single_precision_inverse_transform(frac, inside):
    e_store, e_fft = _errors(frac)
    print(f"sources at {frac} x the half field: complex64 storage {e_store:.1e}, single-precision inverse FFT {e_fft:.1e}")
    assert e_store < 1e-6, "rounding the stored subgrid to complex64 is harmless"
    if inside:
        assert e_fft < 1e-5
    else:
        assert e_fft > 1e-5, "a single-precision inverse transform cannot hold the bar out here"
