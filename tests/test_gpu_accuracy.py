"""Accuracy against kernel padding and subgrid size (the shape of PAPER.md Fig. 3,
:289-313, on synthetic sky: the paper's MWA data are not available).

For each (L, P): point sources at full-image pixels, visibilities from the measurement equation in fp64
(Eq. 1 :45, identity A-terms), then
  fp64: the numpy oracle grids them and its closure images them               (what the method allows)
  fp32: the CUDA path (idg_grid -> idg_grid_to_image on cuda:0, complex64)    (what this library delivers)
and the recovered flux at the source pixels, after the caller's 1 / (T_full n_vis), is compared with the
truth.  The Kaiser-Bessel taper of the synthetic inputs (R15: beta = pi P / 2) sets the fp64 curve; the
fp32 curve follows it down to the single-precision floor.

As a test (`-m gpu`) it runs three of the cases and asserts the shape of the curve; run as a module it writes the
whole table:

    python -m tests.test_gpu_accuracy > profiles/accuracy_sweep_r02.md      (on the GPU box)

It also holds the accuracy check that needs the fp64 CUDA kernels: the fp32 gridders against
the fp64 gridder on ALL 56 896 subgrids of config 2, a size the numpy oracle cannot reach.
Test infrastructure: it imports the oracle, so it lives under tests/.
"""
import os
import sys

import numpy as np
import pytest
import torch

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

import synth  # noqa: E402
from oracle import idg_oracle as orc  # noqa: E402
from tests.util import oracle_params  # noqa: E402

CASES = [(32, 4), (32, 8), (32, 12), (64, 8), (64, 12), (64, 16), (64, 20), (96, 12), (96, 18), (96, 24)]
if os.environ.get("IDG_SWEEP_CASES"):                    # e.g. "64,12;96,18"
    CASES = [tuple(int(v) for v in c.split(",")) for c in os.environ["IDG_SWEEP_CASES"].split(";")]


def one_case(idg, L, P, n_src=6, seed=17):
    cfg = synth.scaled(synth.get_config(2), n_stations=10, n_times=16, n_chan=8, grid_size=1024, cell_arcsec=120.0,
                       subgrid_size=L, padding=P)
    Ng = cfg.grid_size
    obs = synth.make_observation(cfg, vis=None, with_aterms=False)
    rng = np.random.default_rng(seed)
    jy = Ng // 2 + rng.integers(-Ng // 5, Ng // 5, n_src)
    jx = Ng // 2 + rng.integers(-Ng // 5, Ng // 5, n_src)
    flux = rng.uniform(1.0, 10.0, n_src)
    l0 = (jx - Ng // 2) * cfg.image_size / Ng
    m0 = (jy - Ng // 2) * cfg.image_size / Ng
    n0 = orc.nprime(l0, m0)
    kappa = obs.freqs / 299792458.0
    u = obs.uvw[:, 0:1] * kappa[None, :]
    v = obs.uvw[:, 1:2] * kappa[None, :]
    w = obs.uvw[:, 2:3] * kappa[None, :]
    vv = np.zeros(u.shape, np.complex128)
    for s in range(n_src):
        vv += flux[s] * np.exp(-2j * np.pi * (u * l0[s] + v * m0[s] + w * n0[s]))
    vis = np.zeros((cfg.n_rows, cfg.n_chan, 4), np.complex128)
    vis[..., 0] = vv
    vis[..., 3] = vv
    eye = np.zeros((cfg.n_stations, cfg.n_intervals, L, L, 2, 2), np.complex64)
    eye[..., 0, 0] = eye[..., 1, 1] = 1.0
    k1 = synth.kaiser_bessel_1d(L, P)
    taper64 = np.outer(k1, k1)                             # the oracle takes the taper unrounded
    taper = taper64.astype(np.float32)
    t1 = synth.taper_full_1d(Ng, P)
    # the truth at the source pixels: every source contributes its own dirty-beam sidelobes to the others, so
    # the reference is the direct imaging sum of the same visibilities, not the bare flux
    truth = np.zeros(n_src)
    for s in range(n_src):
        truth[s] = np.real(np.sum(vv * np.exp(2j * np.pi * (u * l0[s] + v * m0[s] + w * n0[s])))) / cfg.n_vis

    par = oracle_params(cfg)
    sub, dropped = orc.plan(par, obs.uvw, obs.freqs, cfg.n_baselines)
    assert dropped == 0
    G = orc.grid(par, sub, obs.uvw, obs.freqs, vis, obs.baselines, eye, taper64)
    wl_min, _ = orc.layer_range(sub)
    e64 = 0.0
    for s in range(n_src):
        est = orc.image_at_pixels(par, G, wl_min, [jy[s]], [jx[s]])[0, 0, 0] / (t1[jy[s]] * t1[jx[s]]) / cfg.n_vis
        e64 = max(e64, abs(est.real - truth[s]) / flux.max())

    dev = "cuda:0"
    to = lambda a: torch.from_numpy(np.ascontiguousarray(a)).to(dev)  # noqa: E731
    e32 = {}
    for name, variant in (("simt", idg.VARIANT_SIMT), ("tensor", idg.VARIANT_TENSOR)):
        plan = idg.plan_from_config(cfg, obs.uvw, obs.freqs, obs.baselines, gridder_variant=variant)
        cnt = plan.counts()
        d_grid = torch.zeros((cnt.n_wlayers, 4, Ng, Ng), dtype=torch.complex64, device=dev)
        ws = torch.empty(max(plan.workspace_bytes(), plan.closure_workspace_bytes()), dtype=torch.uint8, device=dev)
        idg.grid(plan, to(vis.astype(np.complex64)), to(eye), to(taper), d_grid, ws)
        d_img = torch.zeros((4, Ng, Ng), dtype=torch.complex64, device=dev)
        idg.grid_to_image(plan, d_grid, d_img, ws, corr=to((1.0 / (np.outer(t1, t1) * cfg.n_vis)).astype(np.float32)))
        img = d_img.cpu().numpy()
        e32[name] = max(abs(img[0, jy[s], jx[s]].real - truth[s]) / flux.max() for s in range(n_src))
    return len(sub), e64, e32["simt"], e32["tensor"]


@pytest.mark.gpu
def test_error_falls_with_padding_down_to_the_fp32_floor(idg):
    """Shape of PAPER.md Fig. 3 (:299): the method's own (fp64) error falls by orders of magnitude with the padding;
    the fp32 path follows it down to a floor near the paper's own single-precision figure (6e-6, :313)."""
    rows = {(L, P): one_case(idg, L, P) for L, P in ((32, 4), (32, 12), (64, 20))}
    e64 = [rows[k][1] for k in ((32, 4), (32, 12), (64, 20))]
    assert e64[0] > 30 * e64[1] > 30 * 30 * e64[2], e64
    for (L, P), (_, m64, simt, tensor) in rows.items():
        assert simt <= max(3.0 * m64, 3e-6) and tensor <= max(3.0 * m64, 3e-6), (L, P, m64, simt, tensor)


@pytest.mark.gpu
@pytest.mark.parametrize("variant", ["simt", "tensor"])
def test_fp32_gridders_against_fp64_on_every_subgrid_of_config2(idg, variant):
    """accuracy at a size the numpy oracle cannot reach.  The fp64 CUDA gridder (itself within
    1e-11 of the oracle, tests/test_gpu_parity.py::test_fp64_direct_sums) is the reference for the fp32 gridders
    on ALL 56 896 subgrids of BASELINE.json configs[1]: the worst normalised error over every subgrid."""
    dev = "cuda:0"
    cfg = synth.get_config(2)
    obs = synth.make_observation(cfg, vis="hash")
    plan = idg.plan_from_config(cfg, obs.uvw, obs.freqs, obs.baselines,
                                gridder_variant={"simt": idg.VARIANT_SIMT, "tensor": idg.VARIANT_TENSOR}[variant])
    n, L = plan.counts().n_subgrids, cfg.subgrid_size
    to = lambda a: torch.from_numpy(np.ascontiguousarray(a)).to(dev)  # noqa: E731
    d_vis, d_at, d_tp = to(obs.vis), to(obs.aterms), to(obs.taper)
    worst, mean, chunk = 0.0, 0.0, 8192
    for first in range(0, n, chunk):
        count = min(chunk, n - first)
        o64 = torch.empty((count, 4, L, L), dtype=torch.complex128, device=dev)
        o32 = torch.empty((count, 4, L, L), dtype=torch.complex64, device=dev)
        idg.grid_subgrids_f64(plan, first, count, d_vis, d_at, d_tp, o64)
        idg.grid_subgrids(plan, first, count, d_vis, d_at, d_tp, o32, stage=idg.STAGE_GRIDDER)
        err = (o32.to(torch.complex128) - o64).abs().reshape(count, -1).amax(dim=1) / o64.abs().reshape(count, -1).amax(dim=1)
        worst = max(worst, float(err.max()))
        mean += float(err.sum())
    print(f"config 2, all {n} subgrids, {variant} gridder vs fp64 gridder: worst {worst:.2e}, mean {mean / n:.2e}")
    assert worst <= 1e-5


def main():
    from paper_2502_17789_b200 import build
    build.build()
    import paper_2502_17789_b200 as idg
    print("# Accuracy against padding and subgrid size (tests/test_gpu_accuracy.py)\n")
    print("Command (GPU box): `python -m tests.test_gpu_accuracy > profiles/accuracy_sweep_r02.md`.  10 stations, "
          "16 x 2 s, 8 channels, grid 1024 x 1024 at 120 arcsec, 6 point sources of 1-10 Jy at image pixels, "
          "Kaiser-Bessel taper beta = pi P / 2.  Error = max over the sources of |recovered - direct sum| / "
          "brightest flux, the direct sum being the imaging equation evaluated on the same visibilities in "
          "fp64.\n")
    print("| L | P | subgrids | fp64 oracle | CUDA fp32, SIMT gridder | CUDA fp32, tensor-core gridder |")
    print("|---|---|---|---|---|---|")
    for L, P in CASES:
        n, e64, es, et = one_case(idg, L, P)
        print(f"| {L} | {P} | {n} | {e64:.1e} | {es:.1e} | {et:.1e} |", flush=True)
    print("\nReading: the fp64 column is the method's own error (taper aliasing), falling by orders of magnitude "
          "with the padding as in the paper's Fig. 3 (`PAPER.md:299`); the fp32 columns follow it down to the "
          "single-precision floor (the paper's fp32 peak error is 43 uJy on 6.9 Jy = 6e-6, `:313`), where more "
          "padding buys nothing.  The SIMT gridder's floor is 3e-7-7e-7: its rounding errors are random and "
          "average down over subgrids.  The tensor-core gridder's floor is 0.8e-6-1.1e-6: the tensor core's fp32 "
          "accumulation truncates, a bias that is coherent across subgrids (24 MMAs per accumulator with the fp16 "
          "operands; the earlier split-tf32 operands, 48 MMAs, gave 1.8e-6; DESIGN.md \"Tensor-core gridder\", "
          "Precision).")


if __name__ == "__main__":
    main()
