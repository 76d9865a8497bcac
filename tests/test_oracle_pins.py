"""Pins for the fp64 oracle against what the paper and the mathematics fix.

None of these re-types the oracle's formula: each compares against an independent statement --
the measurement equation evaluated by brute force (Eq. 1 :45), the closed-form
gridding kernel (IDG 'effects the same outcome' as convolutional gridding, :35), numpy.fft,
mpmath, or an invariant the paper states in words.
"""
import dataclasses

import numpy as np
import pytest

import synth
from oracle import idg_oracle as orc
from tests.util import inner, oracle_params, random_jones, tiny_config

TWO_PI = 2.0 * np.pi


def _setup(cfg, seed=0, vis="hash", aterm="random"):
    obs = synth.make_observation(cfg, vis=vis, with_aterms=False)
    par = oracle_params(cfg)
    sub, dropped = orc.plan(par, obs.uvw, obs.freqs, cfg.n_baselines)
    rng = np.random.default_rng(seed)
    if aterm == "random":
        A = random_jones(rng, (cfg.n_stations, cfg.n_intervals, cfg.subgrid_size, cfg.subgrid_size))
    else:
        A = np.zeros((cfg.n_stations, cfg.n_intervals, cfg.subgrid_size, cfg.subgrid_size, 2, 2), np.complex64)
        A[..., 0, 0] = 1
        A[..., 1, 1] = 1
    return obs, par, sub, dropped, A, rng


def _brute_force_image(cfg, par, obs, A, taper, sub_mask_rows=None, positive_w=False, power_norm=False):
    """taper[i] * sum_k M_p(l_i) V_k M_q(l_i)^H exp(+2 pi i (u_k l_i + v_k m_i + w_k n'_i)) at the
    L x L subgrid sample directions: the discrete imaging equation with A-terms, evaluated
    visibility by visibility straight from Eq. 1 / Eq. 2 of the paper (no subgrids, no FFT)."""
    L, S = cfg.subgrid_size, cfg.image_size
    ax = (np.arange(L) - L // 2) * S / L
    l = ax[None, :]
    m = ax[:, None]
    n1 = np.sqrt(1.0 - l * l - m * m) - 1.0           # PAPER.md:47 written literally
    kappa = obs.freqs / 299792458.0
    out = np.zeros((L, L, 2, 2), np.complex128)
    for b in range(cfg.n_baselines):
        p, q = obs.baselines[b]
        for t in range(cfg.n_times):
            r = b * cfg.n_times + t
            it = t // cfg.aterm_period
            # PAPER.md:178 (fn 4): a sample with w < 0 may be used as the sample (-u,-v,-w) of the baseline
            # (q, p), whose visibility is V^dagger -- the measurement equation's Hermitian symmetry
            flip = positive_w and obs.uvw[r, 2] < 0
            sgn = -1.0 if flip else 1.0
            Mp = A[q if flip else p, it].astype(np.complex128)
            Mq = A[p if flip else q, it].astype(np.complex128)
            acc = np.zeros((L, L, 2, 2), np.complex128)
            for c in range(cfg.n_chan):
                u, v, w = sgn * obs.uvw[r] * kappa[c]
                ph = np.exp(1j * TWO_PI * (u * l + v * m + w * n1))
                V = obs.vis[r, c].astype(np.complex128).reshape(2, 2)
                if flip:
                    V = V.conj().T
                acc += ph[:, :, None, None] * V[None, None]
            term = Mp @ acc @ np.conj(np.swapaxes(Mq, -1, -2))
            if power_norm:
                # divide by the Frobenius norm of the product of the two maps, per pixel
                prod = Mp @ np.conj(np.swapaxes(Mq, -1, -2))
                term = term / np.linalg.norm(prod, ord="fro", axis=(-2, -1))[:, :, None, None]
            out += term
    return taper[:, :, None, None] * out


@pytest.mark.parametrize("w_step", [0.0, 3.0])
def test_p1_brute_force_with_aterms(w_step):
    """P1 (north_star check 1): IDG closure image at the subgrid sample directions equals the
    A-corrected direct transform exactly -- pins O1-O5: signs, sandwich order, taper, FFT
    centring and 1/L^2, adder placement, w-layer factor."""
    cfg = tiny_config(w_step=w_step, ha_mid_deg=25.0 if w_step > 0 else 0.0)
    obs, par, sub, dropped, A, rng = _setup(cfg, seed=1)
    assert dropped == 0
    taper = rng.uniform(0.2, 1.0, (cfg.subgrid_size, cfg.subgrid_size))   # arbitrary positive taper
    if w_step > 0:
        assert len(np.unique(sub[:, 7])) >= 3, "test must exercise several signed w-layers"
    G = orc.grid(par, sub, obs.uvw, obs.freqs, obs.vis, obs.baselines, A, taper)
    wl_min, W = orc.layer_range(sub)
    L, Ng = cfg.subgrid_size, cfg.grid_size
    j = Ng // 2 + (np.arange(L) - L // 2) * (Ng // L)
    img = orc.image_at_pixels(par, G, wl_min, j, j).reshape(L, L, 2, 2)
    ref = _brute_force_image(cfg, par, obs, A, taper)
    err = np.abs(img - ref).max() / np.abs(ref).max()
    assert err < 1e-12, err


@pytest.mark.parametrize("L,P,tol", [(32, 8, 1e-5), (32, 12, 5e-8)])
def test_p2_point_source_recovery(L, P, tol):
    """P2 (check 2): one source of flux S at a fine pixel, identity A-terms, KB taper:
    the closure image / T_full / n_vis at that pixel returns S (taper-limited)."""
    cfg = tiny_config(subgrid_size=L, padding=P)
    obs, par, sub, dropped, A, rng = _setup(cfg, aterm="identity", vis=None)
    Ng, S = cfg.grid_size, cfg.image_size
    jy, jx, flux = Ng // 2 + 37, Ng // 2 - 22, 3.25
    l0, m0 = (jx - Ng // 2) * S / Ng, (jy - Ng // 2) * S / Ng
    n0 = np.sqrt(1 - l0 * l0 - m0 * m0) - 1
    kappa = obs.freqs / 299792458.0
    uvw = obs.uvw[:, None, :] * kappa[None, :, None]
    v = flux * np.exp(-1j * TWO_PI * (uvw[..., 0] * l0 + uvw[..., 1] * m0 + uvw[..., 2] * n0))
    vis = np.zeros((cfg.n_rows, cfg.n_chan, 4), np.complex128)
    vis[..., 0] = v
    vis[..., 3] = v
    taper = synth.taper_subgrid(cfg).astype(np.float64)
    G = orc.grid(par, sub, obs.uvw, obs.freqs, vis, obs.baselines, A, taper)
    wl_min, _ = orc.layer_range(sub)
    img = orc.image_at_pixels(par, G, wl_min, [jy], [jx])[0, 0]
    t1 = synth.taper_full_1d(Ng, P)
    est = img / (t1[jy] * t1[jx]) / cfg.n_vis
    assert abs(est[0] / flux - 1) < tol and abs(est[3] / flux - 1) < tol, est
    assert abs(est[1]) < tol * flux and abs(est[2]) < tol * flux


@pytest.mark.parametrize("w_step", [0.0, 3.0])
def test_p3_adjoint_identity(w_step):
    """P3 (check 3): <degrid(G;M), V> = <G, grid(V;M^H)> to 1e-12 -- pins O6-O9 against O2-O5."""
    cfg = tiny_config(w_step=w_step, ha_mid_deg=25.0 if w_step > 0 else 0.0)
    obs, par, sub, dropped, A, rng = _setup(cfg, seed=3)
    taper = synth.taper_subgrid(cfg).astype(np.float64)
    wl_min, W = orc.layer_range(sub)
    Ng = cfg.grid_size
    G = rng.standard_normal((W, 4, Ng, Ng)) + 1j * rng.standard_normal((W, 4, Ng, Ng))
    V = obs.vis.astype(np.complex128)
    AH = np.conj(np.swapaxes(A, -1, -2))
    lhs = inner(orc.degrid(par, sub, obs.uvw, obs.freqs, G, obs.baselines, A, taper), V)
    rhs = inner(G, orc.grid(par, sub, obs.uvw, obs.freqs, V, obs.baselines, AH, taper))
    assert abs(lhs - rhs) / abs(lhs) < 1e-12, (lhs, rhs)


@pytest.mark.parametrize("L,P", [(32, 8), (96, 18)])
def test_p4_plain_gridding_kernel(L, P):
    """P4 (check 4): identity A-terms, separable taper, one visibility at pixel offset
    (dx, dy) on its w-plane: Shat[gy,gx] = V K(dy-gy') K(dx-gx'),
    K(D) = 1/L sum_i t[i] exp(2 pi i D (i-L/2)/L) -- the convolution kernel IDG is equivalent to
    (Eq. 2).  Kernel mass sum(Shat) = V T(0) = V."""
    Ng, cell = 256, 1e-3
    par = orc.OracleParams(Ng, L, P, cell, 0.0, 1, 1, 1)
    S = Ng * cell
    freq = 150e6
    kappa = freq / 299792458.0
    x0, y0 = 100, 90
    dx, dy = 3.3, -5.7
    X = (x0 + L // 2 - Ng // 2) + dx
    Y = (y0 + L // 2 - Ng // 2) + dy
    uvw = np.array([[X / S / kappa, Y / S / kappa, 0.0]])
    sub = np.array([0, 0, 1, 0, 1, x0, y0, 0], np.int32)
    V = np.array([[[1.5 - 0.5j, 0.25j, -0.75, 2.0 + 1j]]])
    t = synth.kaiser_bessel_1d(L, P)
    ident = np.zeros((1, 1, L, L, 2, 2)); ident[..., 0, 0] = 1; ident[..., 1, 1] = 1
    _, Shat = orc.grid_subgrid(par, sub, uvw, np.array([freq]), V, np.array([[0, 0]]), ident, np.outer(t, t))
    i = np.arange(L) - L // 2
    K = lambda D: np.array([np.sum(t * np.exp(1j * TWO_PI * d * i / L)) / L for d in np.atleast_1d(D)])
    ref = np.outer(K(dy - i), K(dx - i))[:, :, None] * V.reshape(4)[None, None, :]
    assert np.abs(Shat - ref).max() < 1e-13
    assert np.abs(Shat.sum(axis=(0, 1)) - V.reshape(4) * t[L // 2] ** 2).max() < 1e-12


@pytest.mark.parametrize("L,P,tol", [(32, 8, 2e-5), (32, 12, 1e-7)])
def test_p5_prediction_accuracy(L, P, tol):
    """P5: model = point source; degrid(DFT{I / T_full}) against Eq. 1 evaluated directly
    (pins O6-O9 and the taper reading R4)."""
    cfg = tiny_config(subgrid_size=L, padding=P)
    obs, par, sub, dropped, A, rng = _setup(cfg, aterm="identity", vis=None)
    Ng, S = cfg.grid_size, cfg.image_size
    jy, jx, flux = Ng // 2 - 41, Ng // 2 + 30, 2.0
    t1 = synth.taper_full_1d(Ng, P)
    model = np.zeros((4, Ng, Ng), np.complex128)
    model[0, jy, jx] = model[3, jy, jx] = flux / (t1[jy] * t1[jx])
    wl_min, W = orc.layer_range(sub)
    G = orc.model_to_grid(par, model, wl_min, W)
    taper = synth.taper_subgrid(cfg).astype(np.float64)
    V = orc.degrid(par, sub, obs.uvw, obs.freqs, G, obs.baselines, A, taper)
    l0, m0 = (jx - Ng // 2) * S / Ng, (jy - Ng // 2) * S / Ng
    n0 = np.sqrt(1 - l0 * l0 - m0 * m0) - 1
    uvw = obs.uvw[:, None, :] * (obs.freqs / 299792458.0)[None, :, None]
    ref = flux * np.exp(-1j * TWO_PI * (uvw[..., 0] * l0 + uvw[..., 1] * m0 + uvw[..., 2] * n0))
    assert np.abs(V[..., 0] - ref).max() / flux < tol
    assert np.abs(V[..., 3] - ref).max() / flux < tol
    assert np.abs(V[..., 1]).max() < tol and np.abs(V[..., 2]).max() < tol


@pytest.mark.parametrize("L", [32, 64, 96, 128, 48])
def test_p6_fft_against_numpy(L):
    """P6: centred DFT pair vs numpy.fft with shifts; Parseval; checkerboard identity (even L)."""
    rng = np.random.default_rng(L)
    S = rng.standard_normal((L, L, 4)) + 1j * rng.standard_normal((L, L, 4))
    F = orc.subgrid_fft(S)
    ref = np.fft.fftshift(np.fft.fft2(np.fft.ifftshift(S, axes=(0, 1)), axes=(0, 1)), axes=(0, 1)) / (L * L)
    assert np.abs(F - ref).max() < 1e-13
    Bk = orc.subgrid_ifft(S)
    refi = np.fft.fftshift(np.fft.ifft2(np.fft.ifftshift(S, axes=(0, 1)), axes=(0, 1)), axes=(0, 1))
    assert np.abs(Bk - refi).max() < 1e-13
    assert abs(np.sum(np.abs(F) ** 2) * L * L - np.sum(np.abs(S) ** 2)) < 1e-9 * np.sum(np.abs(S) ** 2)
    # round trip carries 1/L^2 (R2: one factor 1/L^2 in each direction)
    assert np.abs(orc.subgrid_ifft(orc.subgrid_fft(S)) * L * L - S).max() < 1e-12
    chk = (-1.0) ** (np.arange(L)[:, None] + np.arange(L)[None, :])
    if L % 4 == 0:
        ref2 = chk[:, :, None] * np.fft.fft2(chk[:, :, None] * S, axes=(0, 1)) / (L * L)
        assert np.abs(F - ref2).max() < 1e-13


def _check_plan_invariants(cfg, obs, par, sub, dropped):
    L, P, Ng, S = cfg.subgrid_size, cfg.padding, cfg.grid_size, cfg.image_size
    kappa = obs.freqs / 299792458.0
    cover = np.zeros((cfg.n_rows, cfg.n_chan), np.int32)
    for s in sub:
        b, t0, nt, c0, nc, x0, y0, wl = (int(v) for v in s)
        assert nt >= 1 and nc >= 1
        assert t0 // cfg.aterm_period == (t0 + nt - 1) // cfg.aterm_period       # one interval (R6)
        assert 0 <= x0 and 0 <= y0 and x0 + L <= Ng and y0 + L <= Ng             # box inside grid
        r0 = b * cfg.n_times + t0
        cover[r0:r0 + nt, c0:c0 + nc] += 1
        rows = obs.uvw[r0:r0 + nt]
        if par.positive_w:
            neg = rows[:, 2] < 0
            assert neg.all() or not neg.any(), "a subgrid mixes conjugated and plain rows"
            rows = np.where(neg[:, None], -rows, rows)                            # fn 4: (u,v,w) -> -(u,v,w)
            assert wl >= 0, "positive_w must leave no negative w-layer"
        uvw = rows[:, None, :] * kappa[None, c0:c0 + nc, None]
        X, Y = uvw[..., 0] * S, uvw[..., 1] * S
        cx, cy = x0 + L // 2 - Ng // 2, y0 + L // 2 - Ng // 2
        # ALL members (not only the corners) within the usable span (R8)
        assert np.abs(X - cx).max() <= (L - P) / 2 + 1e-9
        assert np.abs(Y - cy).max() <= (L - P) / 2 + 1e-9
        if cfg.w_step > 0:
            w0 = (wl + 0.5) * cfg.w_step
            assert np.abs(uvw[..., 2] - w0).max() <= cfg.w_step / 2 + 1e-9        # |w - w0| <= w_max
        else:
            assert wl == 0
    assert cover.max() <= 1                                                       # exactly one subgrid (:70)
    assert int((cover == 0).sum()) == dropped
    key = [tuple(int(v) for v in (s[7], s[0], s[1], s[3])) for s in sub]
    assert key == sorted(key)


@pytest.mark.parametrize("which", ["cfg1", "tiny_w", "cfg3_small", "drops"])
def test_p7_planner_invariants(which):
    """P7: every visibility in exactly one subgrid or counted dropped; members inside the usable
    span; one interval / baseline / layer per subgrid; boxes inside the grid; sorted order."""
    if which == "cfg1":
        cfg = synth.get_config(1)
    elif which == "tiny_w":
        cfg = tiny_config(w_step=3.0, ha_mid_deg=25.0, n_chan=16, chan_width_hz=2e6)
    elif which == "cfg3_small":
        cfg = synth.scaled(synth.get_config(3), n_stations=10, n_times=24, n_chan=384)
    else:
        cfg = tiny_config(cell_arcsec=400.0)      # uv coverage larger than the grid -> drops
    obs = synth.make_observation(cfg, vis=None, with_aterms=False)
    par = oracle_params(cfg)
    sub, dropped = orc.plan(par, obs.uvw, obs.freqs, cfg.n_baselines)
    if which == "drops":
        assert dropped > 0
    elif which == "cfg1":
        assert sub.shape[0] == 56 and dropped == 0          # SURVEY probe A.5
    _check_plan_invariants(cfg, obs, par, sub, dropped)


def test_p8_adder_splitter():
    """P8: <adder(S), G> = <S, splitter(G)>; integer-valued subgrids sum order-independently and
    match np.add.at exactly."""
    rng = np.random.default_rng(8)
    Ng, L, W = 128, 32, 2
    subs = np.array([[0, 0, 1, 0, 1, x, y, wl] for x, y, wl in
                     [(0, 0, 0), (10, 5, 0), (12, 7, 0), (96, 96, 1), (12, 7, 1), (50, 0, 0)]], np.int32)
    S = [rng.integers(-50, 50, (L, L, 4)) + 1j * rng.integers(-50, 50, (L, L, 4)) for _ in subs]
    G = np.zeros((W, 4, Ng, Ng), np.complex128)
    for s, sub in zip(S, subs):
        orc.adder(G, s.astype(np.complex128), sub, 0)
    ref = np.zeros_like(G)
    for s, sub in reversed(list(zip(S, subs))):
        gy, gx = np.meshgrid(np.arange(L), np.arange(L), indexing="ij")
        for p in range(4):
            np.add.at(ref[sub[7], p], (sub[6] + gy, sub[5] + gx), s[:, :, p])
    assert np.array_equal(G, ref)
    H = rng.standard_normal(G.shape) + 1j * rng.standard_normal(G.shape)
    lhs = inner(G, H)
    rhs = sum(inner(s, orc.splitter(H, sub, L, 0)) for s, sub in zip(S, subs))
    assert abs(lhs - rhs) < 1e-9 * abs(lhs)


def test_p9_nprime_extended_precision():
    """P9: n' = sqrt(1-l^2-m^2) - 1 in the cancellation-free form, against 50-digit mpmath."""
    import mpmath as mp
    mp.mp.dps = 50
    for l, m in [(1e-9, 0.0), (3e-5, -2e-5), (1e-3, 1e-3), (0.05, -0.07), (0.3, 0.4), (0.0, 0.0)]:
        ref = mp.sqrt(1 - mp.mpf(l) ** 2 - mp.mpf(m) ** 2) - 1
        got = float(orc.nprime(np.float64(l), np.float64(m)))
        assert abs(got - float(ref)) <= 2 * np.spacing(abs(float(ref))) + 1e-300


def test_subgrid_centre_and_phase_signs():
    """A visibility exactly on a master-grid pixel deposits T(0) = 1 x its value on that pixel and
    nothing elsewhere when the taper is flat (R2), at the pixel the planner's X = u*S names."""
    Ng, L, cell = 128, 32, 2e-3
    par = orc.OracleParams(Ng, L, 0, cell, 0.0, 1, 1, 1)
    S, freq = Ng * cell, 100e6
    kappa = freq / 299792458.0
    px, py = 70, 49                                   # absolute master-grid pixel (x, y)
    uvw = np.array([[(px - Ng // 2) / S / kappa, (py - Ng // 2) / S / kappa, 0.0]])
    sub, dropped = orc.plan(par, uvw, np.array([freq]), 1)
    assert dropped == 0 and sub.shape[0] == 1
    ident = np.zeros((1, 1, L, L, 2, 2)); ident[..., 0, 0] = 1; ident[..., 1, 1] = 1
    V = np.array([[[1 + 2j, 3 - 1j, -2j, 0.5]]])
    G = orc.grid(par, sub, uvw, np.array([freq]), V, np.array([[0, 0]]), ident, np.ones((L, L)))
    ref = np.zeros_like(G)
    ref[0, :, py, px] = V.reshape(4)
    assert np.abs(G - ref).max() < 1e-12


# ---------------------------------------------------------------------------------------------
# P11  w >= 0 by conjugation (footnote 4; R21)
# ---------------------------------------------------------------------------------------------
def _dagger_image(img):
    return np.conj(np.swapaxes(img, -1, -2))


def test_p11_positive_w_brute_force_and_symmetry():
    """With positive_w the closure image equals the direct transform of the conjugated samples
    ((-u,-v,-w), baseline (q,p), V^dagger for every row with w < 0), all layers are >= 0 and fewer than with
    signed layers, and the Hermitian part of the image -- all a Hermitian sky can populate -- is unchanged."""
    cfg = tiny_config(w_step=3.0, ha_mid_deg=25.0)
    obs, par, sub, dropped, A, rng = _setup(cfg, seed=4)
    assert (obs.uvw[:, 2] < 0).any() and (obs.uvw[:, 2] > 0).any(), "need both signs of w"
    par_c = dataclasses.replace(par, positive_w=True)
    sub_c, dropped_c = orc.plan(par_c, obs.uvw, obs.freqs, cfg.n_baselines)
    assert dropped_c == 0 and sub_c[:, 7].min() >= 0
    assert orc.layer_range(sub_c)[1] < orc.layer_range(sub)[1], "fewer w-layers of master grid are needed"
    _check_plan_invariants(cfg, obs, par_c, sub_c, dropped_c)
    taper = rng.uniform(0.2, 1.0, (cfg.subgrid_size, cfg.subgrid_size))
    L, Ng = cfg.subgrid_size, cfg.grid_size
    j = Ng // 2 + (np.arange(L) - L // 2) * (Ng // L)
    G_c = orc.grid(par_c, sub_c, obs.uvw, obs.freqs, obs.vis, obs.baselines, A, taper)
    wl_min_c, _ = orc.layer_range(sub_c)
    img_c = orc.image_at_pixels(par_c, G_c, wl_min_c, j, j).reshape(L, L, 2, 2)
    ref_c = _brute_force_image(cfg, par_c, obs, A, taper, positive_w=True)
    assert np.abs(img_c - ref_c).max() / np.abs(ref_c).max() < 1e-12
    # Hermitian part: the same image as without the option
    G = orc.grid(par, sub, obs.uvw, obs.freqs, obs.vis, obs.baselines, A, taper)
    wl_min, _ = orc.layer_range(sub)
    img = orc.image_at_pixels(par, G, wl_min, j, j).reshape(L, L, 2, 2)
    h, h_c = img + _dagger_image(img), img_c + _dagger_image(img_c)
    assert np.abs(h - h_c).max() / np.abs(h).max() < 1e-12
    assert np.abs(img - img_c).max() / np.abs(img).max() > 1e-3, "the option must change something"


def test_p11_positive_w_prediction_is_the_real_adjoint():
    """The conjugation V -> V^dagger is conjugate-linear, so with positive_w the pair (degrid(.;M), grid(.;M^H))
    is adjoint for the REAL inner product Re<a,b> (which is what an imaging major cycle minimises), and the
    imaginary parts of the two sides are opposite on the conjugated rows only.  Pins O6-O9 with the option."""
    cfg = tiny_config(w_step=3.0, ha_mid_deg=25.0)
    obs, par, sub, dropped, A, rng = _setup(cfg, seed=6)
    par_c = dataclasses.replace(par, positive_w=True)
    sub_c, _ = orc.plan(par_c, obs.uvw, obs.freqs, cfg.n_baselines)
    taper = synth.taper_subgrid(cfg).astype(np.float64)
    wl_min, W = orc.layer_range(sub_c)
    Ng = cfg.grid_size
    G = rng.standard_normal((W, 4, Ng, Ng)) + 1j * rng.standard_normal((W, 4, Ng, Ng))
    V = obs.vis.astype(np.complex128)
    AH = np.conj(np.swapaxes(A, -1, -2))
    pred = orc.degrid(par_c, sub_c, obs.uvw, obs.freqs, G, obs.baselines, A, taper)
    lhs = inner(pred, V)
    rhs = inner(G, orc.grid(par_c, sub_c, obs.uvw, obs.freqs, V, obs.baselines, AH, taper))
    assert abs(lhs.real - rhs.real) / abs(lhs) < 1e-12, (lhs, rhs)
    # row by row: plain rows obey the complex identity, conjugated rows its complex conjugate
    neg = np.repeat(obs.uvw[:, 2] < 0, cfg.n_chan).reshape(cfg.n_rows, cfg.n_chan)
    Vp, Vn = np.where(neg[..., None], 0, V), np.where(neg[..., None], V, 0)
    for Vs, conj in ((Vp, False), (Vn, True)):
        a = inner(pred, Vs)
        b = inner(G, orc.grid(par_c, sub_c, obs.uvw, obs.freqs, Vs, obs.baselines, AH, taper))
        assert abs(a - (np.conj(b) if conj else b)) / abs(a) < 1e-12


def test_p11_positive_w_predicts_a_hermitian_sky():
    """Prediction with positive_w from a physical (Hermitian-brightness) point source equals Eq. 1 evaluated
    directly, like P5, on every row -- conjugated or not -- to the taper-limited tolerance."""
    L, P, tol = 32, 12, 1e-7
    cfg = tiny_config(subgrid_size=L, padding=P, w_step=3.0, ha_mid_deg=25.0)
    obs, par, sub, dropped, A, rng = _setup(cfg, aterm="identity", vis=None)
    par_c = dataclasses.replace(par, positive_w=True)
    sub_c, _ = orc.plan(par_c, obs.uvw, obs.freqs, cfg.n_baselines)
    Ng, S = cfg.grid_size, cfg.image_size
    jy, jx = Ng // 2 - 41, Ng // 2 + 30
    I, Q, U, Vs = 2.0, 0.3, -0.4, 0.25                      # Stokes -> Hermitian brightness matrix
    B = np.array([I + Q, U + 1j * Vs, U - 1j * Vs, I - Q])
    t1 = synth.taper_full_1d(Ng, P)
    model = np.zeros((4, Ng, Ng), np.complex128)
    model[:, jy, jx] = B / (t1[jy] * t1[jx])
    wl_min, W = orc.layer_range(sub_c)
    G = orc.model_to_grid(par_c, model, wl_min, W)
    taper = synth.taper_subgrid(cfg).astype(np.float64)
    V = orc.degrid(par_c, sub_c, obs.uvw, obs.freqs, G, obs.baselines, A, taper)
    l0, m0 = (jx - Ng // 2) * S / Ng, (jy - Ng // 2) * S / Ng
    n0 = np.sqrt(1 - l0 * l0 - m0 * m0) - 1
    uvw = obs.uvw[:, None, :] * (obs.freqs / 299792458.0)[None, :, None]
    ph = np.exp(-1j * TWO_PI * (uvw[..., 0] * l0 + uvw[..., 1] * m0 + uvw[..., 2] * n0))
    ref = ph[..., None] * B[None, None, :]
    assert np.abs(V - ref).max() / I < tol


# ---------------------------------------------------------------------------------------------
# P12  power normalisation by the Frobenius norm (section 3.3; R22)
# ---------------------------------------------------------------------------------------------
def test_p12_power_norm_brute_force():
    """With power_norm every visibility's contribution to the image is divided, per pixel, by the Frobenius norm
    of M_p M_q^H of its baseline and interval (numpy.linalg.norm on the explicit product)."""
    cfg = tiny_config()
    obs, par, sub, dropped, A, rng = _setup(cfg, seed=9)
    par_n = dataclasses.replace(par, power_norm=True)
    taper = rng.uniform(0.2, 1.0, (cfg.subgrid_size, cfg.subgrid_size))
    G = orc.grid(par_n, sub, obs.uvw, obs.freqs, obs.vis, obs.baselines, A, taper)
    wl_min, _ = orc.layer_range(sub)
    L, Ng = cfg.subgrid_size, cfg.grid_size
    j = Ng // 2 + (np.arange(L) - L // 2) * (Ng // L)
    img = orc.image_at_pixels(par_n, G, wl_min, j, j).reshape(L, L, 2, 2)
    ref = _brute_force_image(cfg, par_n, obs, A, taper, power_norm=True)
    assert np.abs(img - ref).max() / np.abs(ref).max() < 1e-12
    # the factor itself: sqrt of the sum of the squared singular values of the product
    Mp, Mq = A[1, 0].astype(np.complex128), A[4, 0].astype(np.complex128)
    sv = np.linalg.svd(Mp @ np.conj(np.swapaxes(Mq, -1, -2)), compute_uv=False)
    assert np.abs(orc.power_norm_factor(Mp, Mq) * np.sqrt((sv ** 2).sum(-1)) - 1).max() < 1e-13


def test_p12_power_norm_correction_is_exact_for_a_shared_aterm():
    """'The final image must then be corrected by the weighted average of this normalisation factor across all
    subgrids': when every station and interval shares one A-term map the average IS the factor,
    so the corrected image equals the un-normalised one exactly; with different maps the weights are the
    subgrids' visibility counts."""
    cfg = tiny_config()
    obs, par, sub, dropped, A, rng = _setup(cfg, seed=10)
    A_shared = np.broadcast_to(A[0:1, 0:1], A.shape).copy()
    par_n = dataclasses.replace(par, power_norm=True)
    taper = synth.taper_subgrid(cfg).astype(np.float64)
    L, Ng = cfg.subgrid_size, cfg.grid_size
    j = Ng // 2 + (np.arange(L) - L // 2) * (Ng // L)
    wl_min, _ = orc.layer_range(sub)
    img = orc.image_at_pixels(par, orc.grid(par, sub, obs.uvw, obs.freqs, obs.vis, obs.baselines, A_shared, taper),
                              wl_min, j, j)
    img_n = orc.image_at_pixels(par_n, orc.grid(par_n, sub, obs.uvw, obs.freqs, obs.vis, obs.baselines, A_shared, taper),
                                wl_min, j, j)
    avg = orc.power_norm_average(par_n, sub, obs.uvw, obs.baselines, A_shared)
    assert np.abs(img_n / avg[:, :, None] - img).max() / np.abs(img).max() < 1e-12
    # general maps: the average weighs each subgrid's factor by its visibility count
    avg2 = orc.power_norm_average(par_n, sub, obs.uvw, obs.baselines, A)
    num, den = np.zeros((L, L)), 0
    for s in sub:
        p, q = obs.baselines[s[0]]
        it = s[1] // cfg.aterm_period
        prod = A[p, it].astype(np.complex128) @ np.conj(np.swapaxes(A[q, it].astype(np.complex128), -1, -2))
        num += int(s[2]) * int(s[4]) / np.linalg.norm(prod, ord="fro", axis=(-2, -1))
        den += int(s[2]) * int(s[4])
    assert den == cfg.n_vis and np.abs(avg2 - num / den).max() < 1e-13


def test_p12_power_norm_breaks_the_adjoint():
    """R16/R22: the normalisation is applied in imaging only, so grid(.; M^H) with power_norm is no longer the
    adjoint of degrid(.; M) -- the documented defect, asserted so that nobody 'fixes' one side silently."""
    cfg = tiny_config()
    obs, par, sub, dropped, A, rng = _setup(cfg, seed=12)
    par_n = dataclasses.replace(par, power_norm=True)
    taper = synth.taper_subgrid(cfg).astype(np.float64)
    wl_min, W = orc.layer_range(sub)
    Ng = cfg.grid_size
    G = rng.standard_normal((W, 4, Ng, Ng)) + 1j * rng.standard_normal((W, 4, Ng, Ng))
    V = obs.vis.astype(np.complex128)
    AH = np.conj(np.swapaxes(A, -1, -2))
    pred_n = orc.degrid(par_n, sub, obs.uvw, obs.freqs, G, obs.baselines, A, taper)
    pred = orc.degrid(par, sub, obs.uvw, obs.freqs, G, obs.baselines, A, taper)
    assert np.array_equal(pred_n, pred), "prediction must not be normalised"
    lhs = inner(pred_n, V)
    rhs = inner(G, orc.grid(par_n, sub, obs.uvw, obs.freqs, V, obs.baselines, AH, taper))
    assert abs(lhs - rhs) / abs(lhs) > 1e-2
