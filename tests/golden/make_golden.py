"""Writes the stored expected values under tests/golden/.  Calls only `oracle/` and the seeded
input generators in `synth/` -- never the CUDA path.

    python tests/golden/make_golden.py

plan_config1.txt : the oracle planner's subgrid table for BASELINE.json configs[0] (reading O1 of
                   DESIGN.md §3; §2.2 :62-72, §3.1 :186-200), one row per subgrid
                   (b t0 nt c0 nc x0 y0 wl).  Integer work: the C++ planner must match bit for bit.
kernel_L32_P8.txt: the closed-form 1-D gridding kernel K(d) = L^-1 sum_i t[i] exp(2 pi i d (i-L/2)/L)
                   of the Kaiser-Bessel taper (R15) at d = -4..4 in steps of 0.25: what one
                   visibility at pixel offset d deposits per axis (PAPER.md :35 "effects the same
                   outcome" as convolutional gridding; pin P4), computed from oracle.subgrid_fft of
                   a one-visibility subgrid.
"""
import os
import sys

import numpy as np

HERE = os.path.dirname(os.path.abspath(__file__))
sys.path.insert(0, os.path.dirname(os.path.dirname(HERE)))

import synth  # noqa: E402
from oracle import idg_oracle as orc  # noqa: E402


def main():
    cfg = synth.get_config(1)
    obs = synth.make_observation(cfg, vis=None, with_aterms=False)
    par = orc.OracleParams(grid_size=cfg.grid_size, subgrid_size=cfg.subgrid_size, padding=cfg.padding,
                           cell_size=cfg.cell_size, w_step=cfg.w_step, n_times=cfg.n_times, n_chan=cfg.n_chan,
                           aterm_period=cfg.aterm_period, comfort=cfg.comfort)
    sub, dropped = orc.plan(par, obs.uvw, obs.freqs, cfg.n_baselines)
    with open(os.path.join(HERE, "plan_config1.txt"), "w") as f:
        f.write(f"# oracle plan of config 1: {len(sub)} subgrids, {dropped} visibilities dropped; columns b t0 nt c0 nc x0 y0 wl\n")
        for row in sub:
            f.write(" ".join(str(int(v)) for v in row) + "\n")

    # one visibility of value 1 at offset d pixels along x from the subgrid centre, identity A-terms:
    # after taper and FFT the row gy = L/2 of the subgrid holds K(d - (gx - L/2)) * K_y(0 - 0)...
    L, P = 32, 8
    S = par.image_size
    t1 = synth.kaiser_bessel_1d(L, P)                 # float64 (taper_subgrid rounds to float32)
    taper = np.outer(t1, t1)
    l = (np.arange(L) - L // 2) * S / L
    with open(os.path.join(HERE, "kernel_L32_P8.txt"), "w") as f:
        f.write("# d  Re K(d)  Im K(d)   (1-D kernel of the L=32, P=8 Kaiser-Bessel taper; see make_golden.py)\n")
        for d in np.arange(-4.0, 4.0001, 0.25):
            du = d / S                                    # d master-grid pixels = d / S wavelengths
            E = np.exp(2j * np.pi * du * l)[None, :] * np.ones((L, 1))
            Sp = (taper * E)[:, :, None]
            Shat = orc.subgrid_fft(Sp)[:, :, 0]
            ky0 = Shat[L // 2, L // 2]                    # = K(d) * K(0)
            k0 = orc.subgrid_fft(taper[:, :, None].astype(np.complex128))[L // 2, L // 2, 0]   # K(0)^2
            K = ky0 / np.sqrt(k0.real)
            f.write(f"{d:+.2f} {K.real:.15e} {K.imag:.15e}\n")


if __name__ == "__main__":
    main()
