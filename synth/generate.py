"""Seeded input generators.  Inputs only -- see package docstring.

Geometry is textbook interferometry (Thompson et al., cited PAPER.md:49) standing in for real
MWA / SKA-Low metadata.  Everything is drawn from numpy.random.default_rng(1000 + config_id).
"""
from __future__ import annotations

import dataclasses
import math

import numpy as np

from .configs import Config

LATITUDE_DEG = -26.7
DECLINATION_DEG = -26.7
EARTH_RATE = 7.2921150e-5          # rad/s
C_LIGHT = 299792458.0


# --------------------------------------------------------------------------------------
# array geometry
# --------------------------------------------------------------------------------------
def _disk(rng, n, diameter):
    r = 0.5 * diameter * np.sqrt(rng.random(n))
    th = 2.0 * np.pi * rng.random(n)
    return r * np.cos(th), r * np.sin(th)


def station_layout(cfg: Config, rng=None):
    """(E, N) station positions in metres."""
    rng = np.random.default_rng(cfg.seed) if rng is None else rng
    if cfg.layout == "disk":
        return _disk(rng, cfg.n_stations, cfg.disk_diameter_m)
    if cfg.layout == "ska":
        n_core = cfg.n_stations // 2
        n_arm = cfg.n_stations - n_core
        e_c, n_c = _disk(rng, n_core, cfg.disk_diameter_m)
        per_arm = -(-n_arm // 3)
        radii = 500.0 * (32500.0 / 500.0) ** (np.arange(per_arm) / max(per_arm - 1, 1))
        i = np.arange(n_arm)
        arm, k = i % 3, i // 3
        r = radii[k]
        th = 2.0 * np.pi * arm / 3.0 + 1.13 * np.log(r / 500.0)
        return np.concatenate([e_c, r * np.cos(th)]), np.concatenate([n_c, r * np.sin(th)])
    raise ValueError(cfg.layout)


def baselines(n_stations: int) -> np.ndarray:
    """int32 [n_bl, 2] station pairs (p < q) in np.triu_indices order."""
    p, q = np.triu_indices(n_stations, k=1)
    return np.stack([p, q], axis=1).astype(np.int32)


def uvw_metres(cfg: Config, east, north) -> np.ndarray:
    """float64 [n_bl * n_times, 3]; row r = b * n_times + t (baseline-major)."""
    lat = math.radians(LATITUDE_DEG)
    dec = math.radians(DECLINATION_DEG)
    X = -north * math.sin(lat)
    Y = east
    Z = north * math.cos(lat)
    bl = baselines(cfg.n_stations)
    bx = (X[bl[:, 1]] - X[bl[:, 0]])[:, None]
    by = (Y[bl[:, 1]] - Y[bl[:, 0]])[:, None]
    bz = (Z[bl[:, 1]] - Z[bl[:, 0]])[:, None]
    t = np.arange(cfg.n_times, dtype=np.float64)
    H = (math.radians(cfg.ha_mid_deg) + (t - (cfg.n_times - 1) / 2.0) * cfg.dt_s * EARTH_RATE)[None, :]
    sH, cH = np.sin(H), np.cos(H)
    sd, cd = math.sin(dec), math.cos(dec)
    u = sH * bx + cH * by
    v = -sd * cH * bx + sd * sH * by + cd * bz
    w = cd * cH * bx - cd * sH * by + sd * bz
    return np.stack([u, v, w], axis=-1).reshape(-1, 3).astype(np.float64)


def channel_freqs(cfg: Config) -> np.ndarray:
    c = np.arange(cfg.n_chan, dtype=np.float64)
    if cfg.freq_is_start:
        return cfg.freq_hz + c * cfg.chan_width_hz
    return cfg.freq_hz + (c - (cfg.n_chan - 1) / 2.0) * cfg.chan_width_hz


# --------------------------------------------------------------------------------------
# sky and visibilities
# --------------------------------------------------------------------------------------
def point_sources(cfg: Config, rng=None):
    """dict(l, m, brightness[n,2,2] complex at nu0, alpha, nu0)."""
    rng = np.random.default_rng(cfg.seed + 17) if rng is None else rng
    n = cfg.n_sources
    if cfg.config_id == 1:
        half = math.sin(math.radians(10.0))          # "within +-10 deg" (aliases outside the field)
        stokes_i = rng.uniform(1.0, 10.0, n)
        alpha = np.zeros(n)
    else:
        half = 0.4 * cfg.image_size                   # inside 0.8x the field
        stokes_i = 10.0 ** rng.uniform(-1.0, 1.0, n)  # log-uniform [0.1, 10] Jy
        alpha = np.full(n, -0.8)
    l = rng.uniform(-half, half, n)
    m = rng.uniform(-half, half, n)
    # random fractional polarisation (<= 30 %) so all four correlations are populated
    q, u_, v_ = (stokes_i * rng.uniform(-0.3, 0.3, n) / math.sqrt(3.0) for _ in range(3))
    B = np.empty((n, 2, 2), np.complex128)
    B[:, 0, 0] = stokes_i + q
    B[:, 0, 1] = u_ + 1j * v_
    B[:, 1, 0] = u_ - 1j * v_
    B[:, 1, 1] = stokes_i - q
    nu0 = float(np.mean(channel_freqs(cfg)))
    return dict(l=l, m=m, brightness=B, alpha=alpha, nu0=nu0)


def source_visibilities(uvw_rows: np.ndarray, freqs: np.ndarray, src: dict) -> np.ndarray:
    """Uncorrupted point-source visibilities, complex64 [n_rows, n_chan, 4] (XX,XY,YX,YY).

    V[r,c] = sum_src B_src(nu_c) exp(-2 pi i (u l + v m + w n'))   (Eq. 1 with A = I).
    This is the *input data* recipe, not part of the method.
    """
    l, m = src["l"], src["m"]
    n1 = -(l * l + m * m) / (1.0 + np.sqrt(1.0 - l * l - m * m))
    kappa = freqs / C_LIGHT
    geo = uvw_rows[:, 0:1] * l[None, :] + uvw_rows[:, 1:2] * m[None, :] + uvw_rows[:, 2:3] * n1[None, :]
    out = np.zeros((uvw_rows.shape[0], freqs.size, 4), np.complex128)
    spec = (freqs[:, None] / src["nu0"]) ** src["alpha"][None, :]            # [chan, src]
    Bf = src["brightness"].reshape(-1, 4)
    for c in range(freqs.size):
        ph = np.exp(-2j * np.pi * kappa[c] * geo)                              # [rows, src]
        out[:, c, :] = (ph * spec[c][None, :]) @ Bf
    return out.astype(np.complex64)


_SM_A = np.uint64(0x9E3779B97F4A7C15)
_SM_B = np.uint64(0xBF58476D1CE4E5B9)
_SM_C = np.uint64(0x94D049BB133111EB)


def hash_visibilities(rows: np.ndarray, n_chan: int, seed: int, n_chan_total: int | None = None,
                      chan0: int = 0) -> np.ndarray:
    """Counter-based pseudo-random visibilities, complex64 [len(rows), n_chan, 4].

    value(row, chan, pol, re/im) = 2*U - 1 with U = top 24 bits of splitmix64(seed, counter)/2^24,
    counter = ((row*n_chan_total + chan)*4 + pol)*2 + reim.  Any subset of rows/channels of the
    full array can be regenerated bit-identically (used to feed the oracle only the sampled
    subgrids of a large workload).  `idg_synth_hash_vis` style device generators must reproduce
    exactly this integer recipe (tests use torch int64 arithmetic, see tests/util.py).
    """
    n_chan_total = n_chan if n_chan_total is None else n_chan_total
    rows = np.asarray(rows, dtype=np.uint64)
    ch = np.arange(chan0, chan0 + n_chan, dtype=np.uint64)
    k = np.arange(8, dtype=np.uint64)
    ctr = ((rows[:, None, None] * np.uint64(n_chan_total) + ch[None, :, None]) * np.uint64(8)
           + k[None, None, :])
    with np.errstate(over="ignore"):
        z = ctr + np.uint64(seed) * _SM_A + _SM_A
        z = (z ^ (z >> np.uint64(30))) * _SM_B
        z = (z ^ (z >> np.uint64(27))) * _SM_C
        z = z ^ (z >> np.uint64(31))
    u24 = (z >> np.uint64(40)).astype(np.float32) * np.float32(2.0 ** -24)
    f = (2.0 * u24 - 1.0).astype(np.float32)
    return np.ascontiguousarray(f).view(np.complex64).reshape(rows.size, n_chan, 4)


# --------------------------------------------------------------------------------------
# taper: separable Kaiser-Bessel, beta = pi P / 2
# --------------------------------------------------------------------------------------
def kaiser_bessel_1d(n: int, padding: int) -> np.ndarray:
    beta = math.pi * padding / 2.0
    x = (np.arange(n, dtype=np.float64) - n // 2) / (n / 2.0)
    return np.i0(beta * np.sqrt(np.maximum(0.0, 1.0 - x * x))) / np.i0(beta)


def taper_subgrid(cfg_or_L, padding: int | None = None) -> np.ndarray:
    """float32 [L, L] taper T = t (x) t sampled at the subgrid pixels."""
    if isinstance(cfg_or_L, Config):
        L, padding = cfg_or_L.subgrid_size, cfg_or_L.padding
    else:
        L = int(cfg_or_L)
    t = kaiser_bessel_1d(L, padding)
    return np.outer(t, t).astype(np.float32)


def taper_full_1d(grid_size: int, padding: int) -> np.ndarray:
    """float64 [Ng]: the same taper function sampled at the full-image pixels (T_full = t (x) t)."""
    return kaiser_bessel_1d(grid_size, padding)


# --------------------------------------------------------------------------------------
# A-terms -- inputs only; parity does not depend on their physics
# --------------------------------------------------------------------------------------
def _subgrid_lm(cfg: Config):
    L = cfg.subgrid_size
    ax = (np.arange(L, dtype=np.float64) - L // 2) * cfg.image_size / L
    return ax[None, :], ax[:, None]                    # l along x, m along y


def _gauss_smooth_periodic(noise: np.ndarray, sigma: float) -> np.ndarray:
    n = noise.shape[-1]
    k = np.fft.fftfreq(n)
    g = np.exp(-2.0 * (np.pi * sigma) ** 2 * (k[None, :] ** 2 + k[:, None] ** 2))
    return np.fft.ifft2(np.fft.fft2(noise) * g).real


def aterms(cfg: Config, rng=None, stations=None) -> np.ndarray:
    """complex64 [n_stations, n_intervals, L, L, 2, 2] Jones maps M[s, it, y, x]."""
    rng = np.random.default_rng(cfg.seed + 29) if rng is None else rng
    L, ns, ni = cfg.subgrid_size, cfg.n_stations, cfg.n_intervals
    out = np.zeros((ns, ni, L, L, 2, 2), np.complex64)
    l, m = _subgrid_lm(cfg)
    lam = C_LIGHT / float(np.mean(channel_freqs(cfg)))
    if cfg.aterm_kind == "fourier":
        x = np.arange(L)[None, :] / L
        y = np.arange(L)[:, None] / L
        for s in range(ns):
            for it in range(ni):
                for j in range(2):
                    for k in range(2):
                        F = np.zeros((L, L), np.complex128)
                        for a in (-1, 0, 1):
                            for b in (-1, 0, 1):
                                c = (rng.standard_normal() + 1j * rng.standard_normal()) / math.sqrt(2.0) / 3.0
                                F += c * np.exp(2j * np.pi * (a * x + b * y))
                        out[s, it, :, :, j, k] = (1.0 if j == k else 0.0) + cfg.screen_rms * F
    elif cfg.aterm_kind == "beam_screen":
        r2 = l * l + m * m
        n = np.sqrt(1.0 - r2)
        h = 0.3
        g = np.sin(2.0 * np.pi * h * n / lam) / math.sin(2.0 * np.pi * h / lam)
        J = np.empty((L, L, 2, 2), np.float64)
        J[..., 0, 0] = g * (1.0 - l * l / (1.0 + n))
        J[..., 0, 1] = g * (-l * m / (1.0 + n))
        J[..., 1, 0] = J[..., 0, 1]
        J[..., 1, 1] = g * (1.0 - m * m / (1.0 + n))
        for s in range(ns):
            noise = rng.standard_normal((ni, L, L))
            for it in range(ni):
                f = _gauss_smooth_periodic(noise[it], L / 8.0) if cfg.screen_smooth else noise[it]
                f = f * (cfg.screen_rms / max(float(np.sqrt(np.mean(f * f))), 1e-30))
                out[s, it] = (J * np.exp(1j * f)[..., None, None]).astype(np.complex64)
    elif cfg.aterm_kind == "array_factor":
        n_el = 256
        lx = l[0] / lam          # [L]
        my = m[:, 0] / lam
        for s in range(ns):
            r = 19.0 * np.sqrt(rng.random(n_el))
            th = 2.0 * np.pi * rng.random(n_el)
            xe, ye = r * np.cos(th), r * np.sin(th)
            Ex = np.exp(2j * np.pi * xe[:, None] * lx[None, :])      # [el, x]
            Ey = np.exp(2j * np.pi * ye[:, None] * my[None, :])      # [el, y]
            for it in range(ni):
                psi = cfg.screen_rms * rng.standard_normal(n_el)
                af = (Ey * np.exp(1j * psi)[:, None]).T @ Ex / n_el  # [y, x]
                out[s, it, :, :, 0, 0] = af
                out[s, it, :, :, 1, 1] = af
    else:
        raise ValueError(cfg.aterm_kind)
    return out


# --------------------------------------------------------------------------------------
# bundle
# --------------------------------------------------------------------------------------
@dataclasses.dataclass
class Observation:
    cfg: Config
    baselines: np.ndarray      # int32 [n_bl, 2]
    uvw: np.ndarray            # float64 [n_rows, 3] metres
    freqs: np.ndarray          # float64 [n_chan]
    vis: np.ndarray | None     # complex64 [n_rows, n_chan, 4]
    aterms: np.ndarray | None  # complex64 [n_st, n_int, L, L, 2, 2]
    taper: np.ndarray          # float32 [L, L]
    sources: dict | None = None


def make_observation(cfg: Config, vis: str | None = "sources", with_aterms: bool = True) -> Observation:
    """Full seeded observation.  vis: "sources" | "hash" | None (caller fills it, e.g. on device)."""
    e, n = station_layout(cfg)
    uvw = uvw_metres(cfg, e, n)
    fr = channel_freqs(cfg)
    src = point_sources(cfg)
    if vis == "sources":
        v = source_visibilities(uvw, fr, src)
    elif vis == "hash":
        v = hash_visibilities(np.arange(cfg.n_rows), cfg.n_chan, cfg.seed)
    elif vis is None:
        v = None
    else:
        raise ValueError(vis)
    A = aterms(cfg) if with_aterms else None
    return Observation(cfg, baselines(cfg.n_stations), uvw, fr, v, A, taper_subgrid(cfg), src)


def source_visibilities_torch(uvw_rows: np.ndarray, freqs: np.ndarray, src: dict, device, chunk_rows: int = 16384):
    """The recipe of `source_visibilities` evaluated with torch fp64 on `device`, in row chunks, for
    the large workloads ("generate them on-device with torch in chunks").
    Returns a torch complex64 tensor [n_rows, n_chan, 4] on `device`.  Input data only."""
    import torch

    l = torch.as_tensor(src["l"], dtype=torch.float64, device=device)
    m = torch.as_tensor(src["m"], dtype=torch.float64, device=device)
    n1 = -(l * l + m * m) / (1.0 + torch.sqrt(1.0 - l * l - m * m))
    kappa = torch.as_tensor(freqs / C_LIGHT, dtype=torch.float64, device=device)
    spec = torch.as_tensor((freqs[:, None] / src["nu0"]) ** src["alpha"][None, :], dtype=torch.float64, device=device)
    Bf = torch.as_tensor(src["brightness"].reshape(-1, 4), dtype=torch.complex128, device=device)
    n_rows = uvw_rows.shape[0]
    out = torch.empty((n_rows, freqs.size, 4), dtype=torch.complex64, device=device)
    for r0 in range(0, n_rows, chunk_rows):
        rows = torch.as_tensor(uvw_rows[r0:r0 + chunk_rows], dtype=torch.float64, device=device)
        geo = rows[:, 0:1] * l[None, :] + rows[:, 1:2] * m[None, :] + rows[:, 2:3] * n1[None, :]   # [rows, src]
        for c in range(freqs.size):
            ang = (-2.0 * math.pi) * kappa[c] * geo
            ph = torch.complex(torch.cos(ang), torch.sin(ang)) * spec[c][None, :]
            out[r0:r0 + chunk_rows, c, :] = (ph @ Bf).to(torch.complex64)
    return out


def hash_visibilities_torch(n_rows: int, n_chan: int, seed: int, device, chunk_rows: int = 1 << 16):
    """`hash_visibilities` for all rows 0..n_rows-1, evaluated with torch int64 arithmetic on `device` in row
    chunks (two's-complement wrap-around = the uint64 recipe; shifts made logical by masking).  Bit-identical to
    the numpy generator (tests/test_synth.py checks sampled rows).  Returns complex64 [n_rows, n_chan, 4]."""
    import torch

    def i64(x):                       # uint64 constant -> the int64 with the same bits
        x = int(x) & 0xFFFFFFFFFFFFFFFF
        return x - (1 << 64) if x >= (1 << 63) else x

    def lsr(z, k):
        return (z >> k) & ((1 << (64 - k)) - 1)

    A, B, C = i64(_SM_A), i64(_SM_B), i64(_SM_C)
    # (seed * A + A) mod 2^64 as a Python integer: torch cannot multiply by it without overflow warnings
    off = i64((int(seed) * int(_SM_A) + int(_SM_A)) & 0xFFFFFFFFFFFFFFFF)
    out = torch.empty((n_rows, n_chan, 4), dtype=torch.complex64, device=device)
    ch = torch.arange(n_chan, dtype=torch.int64, device=device)
    k = torch.arange(8, dtype=torch.int64, device=device)
    for r0 in range(0, n_rows, chunk_rows):
        rows = torch.arange(r0, min(n_rows, r0 + chunk_rows), dtype=torch.int64, device=device)
        ctr = (rows[:, None, None] * n_chan + ch[None, :, None]) * 8 + k[None, None, :]
        z = ctr + off
        z = (z ^ lsr(z, 30)) * B
        z = (z ^ lsr(z, 27)) * C
        z = z ^ lsr(z, 31)
        u24 = lsr(z, 40).to(torch.float32) * (2.0 ** -24)
        f = (2.0 * u24 - 1.0).to(torch.float32).contiguous()
        out[r0:r0 + rows.numel()] = torch.view_as_complex(f.view(rows.numel(), n_chan, 4, 2))
    return out
