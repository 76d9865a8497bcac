"""w-stacking closure on the device against the oracle's closure (Eq. 11
:145-148, Eq. 12 :164-166), and the paper-level pins it enables on GPU output: point-source recovery (P2)
and prediction accuracy (P5) through the whole device chain."""
import numpy as np
import pytest
import torch

import synth
from oracle import idg_oracle as orc
from tests.util import inner, oracle_params

pytestmark = pytest.mark.gpu
DEV = "cuda:0"
TOL = 1e-5


def dev(a):
    return torch.from_numpy(np.ascontiguousarray(a)).to(DEV)


def layered_config():
    return synth.scaled(synth.get_config(3), n_stations=7, n_times=8, n_chan=48, grid_size=512, cell_arcsec=240.0,
                        w_step=4.0, ha_mid_deg=30.0)


@pytest.mark.parametrize("make", [lambda: synth.get_config(1), layered_config], ids=["cfg1", "layers"])
def test_grid_to_image_and_back_match_the_oracle(idg, make):
    cfg = make()
    obs = synth.make_observation(cfg, vis="hash")
    par = oracle_params(cfg)
    plan = idg.plan_from_config(cfg, obs.uvw, obs.freqs, obs.baselines)
    cnt = plan.counts()
    Ng, W = cfg.grid_size, cnt.n_wlayers
    rng = np.random.default_rng(5)
    G = (rng.standard_normal((W, 4, Ng, Ng)) + 1j * rng.standard_normal((W, 4, Ng, Ng))).astype(np.complex64)
    corr = rng.uniform(0.5, 2.0, (Ng, Ng)).astype(np.float32)
    d_img = torch.zeros((4, Ng, Ng), dtype=torch.complex64, device=DEV)
    ws = torch.empty(plan.closure_workspace_bytes(), dtype=torch.uint8, device=DEV)
    d_G = dev(G)
    idg.grid_to_image(plan, d_G, d_img, ws, corr=dev(corr))
    assert torch.equal(torch.view_as_real(d_G).cpu(), torch.view_as_real(torch.from_numpy(G))), "grid not preserved"
    img = d_img.cpu().numpy()
    jy = np.array([0, 1, Ng // 2 - 1, Ng // 2, Ng // 2 + 3, Ng - 1] + rng.integers(0, Ng, 6).tolist())
    jx = np.array([0, 2, Ng // 2, Ng // 2 + 1, Ng - 2, Ng - 1] + rng.integers(0, Ng, 6).tolist())
    ref = orc.image_at_pixels(par, G.astype(np.complex128), cnt.wl_min, jy, jx) * corr[np.ix_(jy, jx)][:, :, None]
    got = np.moveaxis(img[:, jy][:, :, jx], 0, 2)
    scale = np.abs(img).max()
    assert np.abs(got - ref).max() <= TOL * scale, np.abs(got - ref).max() / scale

    # prediction side: the whole [W, 4, Ng, Ng] grid against the oracle
    model = (rng.standard_normal((4, Ng, Ng)) + 1j * rng.standard_normal((4, Ng, Ng))).astype(np.complex64)
    d_out = torch.zeros((W, 4, Ng, Ng), dtype=torch.complex64, device=DEV)
    idg.image_to_grid(plan, dev(model), d_out, corr=dev(corr))
    ref_g = orc.model_to_grid(par, model.astype(np.complex128) * corr[None], cnt.wl_min, W)
    got_g = d_out.cpu().numpy()
    assert np.abs(got_g - ref_g).max() <= TOL * np.abs(ref_g).max()

    # the two are adjoint (no correction): <grid_to_image(G), m> = <G, image_to_grid(m)>
    idg.grid_to_image(plan, d_G, d_img, ws)
    idg.image_to_grid(plan, dev(model), d_out)
    lhs = inner(d_img.cpu().numpy().astype(np.complex128), model.astype(np.complex128))
    rhs = inner(G.astype(np.complex128), d_out.cpu().numpy().astype(np.complex128))
    assert abs(lhs - rhs) / abs(lhs) < 1e-4, (lhs, rhs)


def test_point_source_through_the_device_chain(idg):
    """P2 and P5 on GPU output: visibilities of one point source at a full-image pixel, identity A-terms ->
    idg_grid -> idg_grid_to_image with 1 / (T_full n_vis) recovers the flux at that pixel (taper-limited,
    PAPER.md:291-299); the model image -> idg_image_to_grid -> idg_degrid predicts the same visibilities."""
    cfg = synth.scaled(synth.get_config(2), n_stations=10, n_times=16, grid_size=1024, cell_arcsec=120.0)
    Ng, L, P = cfg.grid_size, cfg.subgrid_size, cfg.padding
    obs = synth.make_observation(cfg, vis=None, with_aterms=False)
    jy, jx, flux = Ng // 2 + 37, Ng // 2 - 91, 3.5
    l0 = (jx - Ng // 2) * cfg.image_size / Ng
    m0 = (jy - Ng // 2) * cfg.image_size / Ng
    n0 = float(orc.nprime(np.float64(l0), np.float64(m0)))
    kappa = obs.freqs / 299792458.0
    u = obs.uvw[:, 0:1] * kappa[None, :]
    v = obs.uvw[:, 1:2] * kappa[None, :]
    w = obs.uvw[:, 2:3] * kappa[None, :]
    vv = flux * np.exp(-2j * np.pi * (u * l0 + v * m0 + w * n0))              # Eq. 1 with A = I
    vis = np.zeros((cfg.n_rows, cfg.n_chan, 4), np.complex64)
    vis[..., 0] = vv
    vis[..., 3] = vv
    eye = np.zeros((cfg.n_stations, cfg.n_intervals, L, L, 2, 2), np.complex64)
    eye[..., 0, 0] = eye[..., 1, 1] = 1.0
    taper = synth.taper_subgrid(cfg)
    t1 = synth.taper_full_1d(Ng, P)
    tfull = np.outer(t1, t1)
    plan = idg.plan_from_config(cfg, obs.uvw, obs.freqs, obs.baselines)
    cnt = plan.counts()
    assert cnt.n_vis_dropped == 0
    d_at, d_tp = dev(eye), dev(taper)
    d_grid = torch.zeros((cnt.n_wlayers, 4, Ng, Ng), dtype=torch.complex64, device=DEV)
    ws = torch.empty(max(plan.workspace_bytes(), plan.closure_workspace_bytes()), dtype=torch.uint8, device=DEV)
    idg.grid(plan, dev(vis), d_at, d_tp, d_grid, ws)
    d_img = torch.zeros((4, Ng, Ng), dtype=torch.complex64, device=DEV)
    idg.grid_to_image(plan, d_grid, d_img, ws, corr=dev((1.0 / (tfull * cfg.n_vis)).astype(np.float32)))
    img = d_img.cpu().numpy()
    est = img[:, jy, jx]
    tol = 2e-5                                            # fp32 path + the taper's aliasing floor at L = 64, P = 12
    assert abs(est[0] / flux - 1) < tol and abs(est[3] / flux - 1) < tol, est
    assert abs(est[1]) < tol * flux and abs(est[2]) < tol * flux
    # brightest pixel of the inner half of the field (1 / T_full blows the edges up)
    q = Ng // 4
    inner_img = np.abs(img[0, q:-q, q:-q])
    assert np.unravel_index(inner_img.argmax(), inner_img.shape) == (jy - q, jx - q)

    # prediction: a delta model at the same pixel, divided by T_full by the caller (R4)
    model = np.zeros((4, Ng, Ng), np.complex64)
    model[0, jy, jx] = model[3, jy, jx] = flux
    idg.image_to_grid(plan, dev(model), d_grid, corr=dev((1.0 / tfull).astype(np.float32)))
    d_out = torch.zeros((cfg.n_rows, cfg.n_chan, 4), dtype=torch.complex64, device=DEV)
    idg.degrid(plan, d_grid, d_at, d_tp, d_out, ws)
    out = d_out.cpu().numpy()
    assert np.abs(out - vis).max() <= 2e-5 * flux, np.abs(out - vis).max() / flux
