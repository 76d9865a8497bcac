"""fp64 CPU oracle for the image-domain-gridding (IDG) hot path.  TEST INFRASTRUCTURE ONLY.

Only `tests/`, `__graft_entry__.smoke()` and `bench.py`'s cpu_baseline / `--impl reference`
legs may import this module.  It shares no code with `paper_2502_17789_b200/` (the CUDA
path) and neither imports the other.  It is deliberately plain and slow: numpy complex128, one
subgrid at a time, the paper's definitions written out with no blocking, fusion or reordering.

Every function cites the passage of /root/reference/PAPER.md (arxiv 2502.17789) it follows;
"R<n>" refers to the readings of silent/ambiguous points listed in DESIGN.md (from SURVEY.md
§8(c)).  Pins: tests/test_oracle_pins.py checks this file against brute-force evaluation of
the measurement equation (P1), point-source recovery (P2), the adjoint identity (P3), the
closed-form gridding kernel (P4), prediction accuracy (P5), numpy.fft (P6), planner
invariants (P7), adder/splitter adjointness (P8), n' in extended precision (P9), the
w >= 0 conjugation against the measurement equation's Hermitian symmetry (P11) and the
power normalisation against an explicit Frobenius norm and its exact-correction case (P12).
Parity unpinned: nothing.

Conventions:
  Ng grid size, cell [rad], S = Ng*cell; L subgrid size; P total kernel padding.
  kappa_c = nu_c / 299792458.0;  row r = b*n_times + t;  u = u_m(r)*kappa_c [wavelengths];
  X = u*S [master-grid pixels from the centre Ng/2].
  subgrid s = (b, t0, nt, c0, nc, x0, y0, wl); cx = x0 + L/2; u0 = (cx - Ng/2)/S;
  w0 = (wl + 1/2)*w_step if w_step > 0 else 0.
  subgrid pixel (y, x): l_x = (x - L/2)*S/L, m_y = (y - L/2)*S/L,
  n' = -(l^2+m^2)/(1+sqrt(1-l^2-m^2))  (= sqrt(1-l^2-m^2) - 1, stable form, R13).
  vis[r, c, 0..3] = (XX, XY, YX, YY) = row-major 2x2 (R14).
"""
from __future__ import annotations

import dataclasses
import math

import numpy as np

C_LIGHT = 299792458.0


@dataclasses.dataclass(frozen=True)
class OracleParams:
    grid_size: int
    subgrid_size: int
    padding: int
    cell_size: float
    w_step: float
    n_times: int
    n_chan: int
    aterm_period: int
    comfort: float = 0.75
    # PAPER.md:178 (footnote 4): force w >= 0 by V(u,v,w) = V(-u,-v,-w)^dagger; reading R21 in DESIGN.md
    positive_w: bool = False
    # PAPER.md:257 (section 3.3): divide the subgrid by the Frobenius norm of M_p M_q^H; reading R22
    power_norm: bool = False

    @property
    def image_size(self) -> float:
        return self.grid_size * self.cell_size


# ======================================================================================
# O1  planner  (§2.2 :62-72, §2.4 :141-143, §3.1 :190-196, §3.3 :255)
# ======================================================================================
def plan(par: OracleParams, uvw_m: np.ndarray, freqs: np.ndarray, n_baselines: int,
         baseline_subset=None):
    """Partition the visibility table of every baseline into subtables = subgrids.

    Single pass per baseline and A-term interval (R6): split the first timestep into channel
    ranges that fit 'comfortably' (R7: span <= comfort*(L-P-1)), then grow each in time until
    the span L-P-1 would be exceeded; only the corners are tested (:196).
    Subgrids snap to a master-grid pixel (:66, R12 round-half-up) and to one w-layer
    (:143, R9: wl = floor(w / w_step)).

    Returns (int32 [n_subgrids, 8] rows (b,t0,nt,c0,nc,x0,y0,wl) sorted by (wl,b,t0,c0),
             n_vis_dropped).
    """
    Ng, L, P = par.grid_size, par.subgrid_size, par.padding
    S = Ng * par.cell_size
    kappa = np.asarray(freqs, np.float64) / C_LIGHT
    span_max = float(L - P - 1)
    comfort_span = par.comfort * span_max
    nT, nC = par.n_times, par.n_chan
    out = []
    dropped = 0
    bls = range(n_baselines) if baseline_subset is None else baseline_subset
    for b in bls:
        rows = np.asarray(uvw_m[b * nT:(b + 1) * nT], np.float64)
        # PAPER.md:178 (fn 4): a row with w < 0 is used as the row (-u,-v,-w) of the swapped baseline
        # (R21); its subgrids then lie in layers wl >= 0.  A subgrid never mixes the two kinds of row.
        FLIP = (rows[:, 2] < 0.0) if par.positive_w else np.zeros(nT, bool)
        rows = np.where(FLIP[:, None], -rows, rows)
        X = (rows[:, 0:1] * kappa[None, :]) * S          # [t, c]  exactly this fp64 order
        Y = (rows[:, 1:2] * kappa[None, :]) * S
        if par.w_step > 0:
            WL = np.floor((rows[:, 2:3] * kappa[None, :]) / par.w_step).astype(np.int64)
        else:
            WL = np.zeros((nT, nC), np.int64)
        n_int = -(-nT // par.aterm_period)
        for it in range(n_int):
            ta = it * par.aterm_period
            tb = min(ta + par.aterm_period, nT)
            work = [(ta, 0, nC - 1)]
            while work:
                t0, lo, hi = work.pop()
                wl0 = WL[t0, lo]
                c1 = lo
                while (c1 + 1 <= hi
                       and max(abs(X[t0, c1 + 1] - X[t0, lo]), abs(Y[t0, c1 + 1] - Y[t0, lo])) <= comfort_span
                       and WL[t0, c1 + 1] == wl0):
                    c1 += 1
                if c1 < hi:
                    work.append((t0, c1 + 1, hi))
                xmin = min(X[t0, lo], X[t0, c1]); xmax = max(X[t0, lo], X[t0, c1])
                ymin = min(Y[t0, lo], Y[t0, c1]); ymax = max(Y[t0, lo], Y[t0, c1])
                n = 1
                while t0 + n < tb:
                    t = t0 + n
                    if WL[t, lo] != wl0 or WL[t, c1] != wl0 or FLIP[t] != FLIP[t0]:
                        break
                    nxmin = min(xmin, X[t, lo], X[t, c1]); nxmax = max(xmax, X[t, lo], X[t, c1])
                    nymin = min(ymin, Y[t, lo], Y[t, c1]); nymax = max(ymax, Y[t, lo], Y[t, c1])
                    if (nxmax - nxmin) > span_max or (nymax - nymin) > span_max:
                        break
                    xmin, xmax, ymin, ymax = nxmin, nxmax, nymin, nymax
                    n += 1
                if t0 + n < tb:
                    work.append((t0 + n, lo, c1))
                cx = int(math.floor((xmin + xmax) / 2.0 + 0.5)) + Ng // 2
                cy = int(math.floor((ymin + ymax) / 2.0 + 0.5)) + Ng // 2
                x0, y0 = cx - L // 2, cy - L // 2
                nc = c1 - lo + 1
                if x0 < 0 or y0 < 0 or x0 + L > Ng or y0 + L > Ng:
                    dropped += n * nc
                    continue
                out.append((int(wl0), b, t0, lo, (b, t0, n, lo, nc, x0, y0, int(wl0))))
    out.sort(key=lambda e: e[:4])
    sub = np.array([e[4] for e in out], np.int32).reshape(-1, 8)
    return sub, dropped


# ======================================================================================
# geometry helpers
# ======================================================================================
def subgrid_lmn(par: OracleParams):
    """(l[x], m[y], n'[y,x]) at the L x L subgrid pixels (R3: no half-pixel offset; the
    subgrid spans the full field S, critically sampled)."""
    L, S = par.subgrid_size, par.image_size
    ax = (np.arange(L, dtype=np.float64) - L // 2) * S / L
    l = ax[None, :]
    m = ax[:, None]
    r2 = l * l + m * m
    n1 = -r2 / (1.0 + np.sqrt(1.0 - r2))
    return ax, ax, n1


def nprime(l, m):
    """n' = sqrt(1-l^2-m^2) - 1 in the cancellation-free form (R13)."""
    r2 = l * l + m * m
    return -r2 / (1.0 + np.sqrt(1.0 - r2))


def subgrid_centre(par: OracleParams, sub):
    """(u0, v0, w0) of a subgrid in wavelengths."""
    Ng, L, S = par.grid_size, par.subgrid_size, par.image_size
    _, _, _, _, _, x0, y0, wl = (int(v) for v in sub)
    u0 = (x0 + L // 2 - Ng // 2) / S
    v0 = (y0 + L // 2 - Ng // 2) / S
    w0 = (wl + 0.5) * par.w_step if par.w_step > 0 else 0.0
    return u0, v0, w0


def subgrid_conjugated(par, sub, uvw_m):
    """True when the subgrid's rows are used in their conjugated form (PAPER.md:178 fn 4, R21):
    the plan asked for w >= 0 and the rows' w is negative (all rows of a subgrid agree, O1)."""
    if not par.positive_w:
        return False
    b, t0 = int(sub[0]), int(sub[1])
    return bool(uvw_m[b * par.n_times + t0][2] < 0.0)


def dagger(V):
    """V^dagger of row-major 2x2 matrices stored as [..., 4] = (XX, XY, YX, YY)."""
    return np.conj(np.asarray(V)[..., [0, 2, 1, 3]])


def _subgrid_relative_uvw(par, sub, uvw_m, freqs):
    b, t0, nt, c0, nc = (int(v) for v in sub[:5])
    kappa = np.asarray(freqs[c0:c0 + nc], np.float64) / C_LIGHT
    r0 = b * par.n_times + t0
    rows = np.asarray(uvw_m[r0:r0 + nt], np.float64)
    if subgrid_conjugated(par, sub, uvw_m):
        rows = -rows                                     # V(u,v,w) = V(-u,-v,-w)^dagger
    u0, v0, w0 = subgrid_centre(par, sub)
    du = rows[:, 0:1] * kappa[None, :] - u0              # [nt, nc]
    dv = rows[:, 1:2] * kappa[None, :] - v0
    dw = rows[:, 2:3] * kappa[None, :] - w0
    return r0, du.reshape(-1), dv.reshape(-1), dw.reshape(-1)


def _phase(par, du, dv, dw):
    """phi[k, y, x] in cycles (Eq. 10, :133-137)."""
    l, m, n1 = subgrid_lmn(par)
    return (du[:, None, None] * l[None, None, :] + dv[:, None, None] * m[None, :, None]
            + dw[:, None, None] * n1[None, :, :])


# ======================================================================================
# O2  gridder: S[y,x] = sum_k V_k exp(+2 pi i phi)      (Eq. 10 :133-137; 2x2 per :253)
# ======================================================================================
def gridder_subgrid(par, sub, uvw_m, freqs, vis):
    """Raw direct sum for one subgrid -> complex128 [L, L, 4] (before A-term and taper)."""
    b, t0, nt, c0, nc = (int(v) for v in sub[:5])
    r0, du, dv, dw = _subgrid_relative_uvw(par, sub, uvw_m, freqs)
    V = np.asarray(vis[r0:r0 + nt, c0:c0 + nc, :], np.complex128).reshape(nt * nc, 4)
    if subgrid_conjugated(par, sub, uvw_m):
        V = dagger(V)
    E = np.exp(2j * np.pi * _phase(par, du, dv, dw))     # one sum over k, as Eq. 10 is written
    return np.einsum("kyx,kp->yxp", E, V)


# ======================================================================================
# O3 / O8  A-term sandwich and taper:  S' = T * M_p * S * M_q^H   (PAPER.md :156, :251-257; R5)
# ======================================================================================
def aterm_taper(S, Mp, Mq, taper, power_norm=False):
    """S [L,L,4] -> taper[y,x] * M_p[y,x] @ S[y,x] @ M_q[y,x]^H, per pixel (2x2 row-major).
    power_norm (imaging only, R22): the result is divided by || M_p M_q^H ||_F per pixel."""
    L = S.shape[0]
    X = S.reshape(L, L, 2, 2)
    Mp = np.asarray(Mp, np.complex128)
    Mq = np.asarray(Mq, np.complex128)
    Y = np.einsum("yxab,yxbc,yxdc->yxad", Mp, X, np.conj(Mq), optimize=True)
    out = np.asarray(taper, np.float64)[:, :, None, None] * Y
    if power_norm:
        out = out * power_norm_factor(Mp, Mq)[:, :, None, None]
    return out.reshape(L, L, 4)


def power_norm_factor(Mp, Mq):
    """f[y,x] = 1 / || M_p[y,x] M_q[y,x]^H ||_F  ('normalising I-hat by the Frobenius norm of
    the product A_1^-1 (A_2^-1)^dagger'; the maps given ARE the A^-1 of paper-style imaging, R5)."""
    Pm = np.einsum("yxab,yxcb->yxac", np.asarray(Mp, np.complex128), np.conj(np.asarray(Mq, np.complex128)))
    return 1.0 / np.sqrt((np.abs(Pm) ** 2).sum(axis=(2, 3)))


def subgrid_jones(par, sub, baselines, aterms, uvw_m=None):
    """(M_p, M_q) maps of a subgrid: interval it = t0 div aterm_period (R6), stations of b; the two swap
    when the subgrid's rows are conjugated (PAPER.md:178 fn 4, R21; needs uvw_m to tell)."""
    b, t0 = int(sub[0]), int(sub[1])
    it = t0 // par.aterm_period
    p, q = int(baselines[b][0]), int(baselines[b][1])
    if uvw_m is not None and subgrid_conjugated(par, sub, uvw_m):
        p, q = q, p
    return aterms[p, it], aterms[q, it]


def power_norm_average(par, subgrids, uvw_m, baselines, aterms):
    """Weighted average over the subgrids of the normalisation factor, weights = visibilities per subgrid:
    'the final image must then be corrected by the weighted average of this normalisation factor across all
    subgrids' (R22) -> float64 [L, L]."""
    L = par.subgrid_size
    num = np.zeros((L, L), np.float64)
    den = 0.0
    for sub in subgrids:
        Mp, Mq = subgrid_jones(par, sub, baselines, aterms, uvw_m)
        n = float(int(sub[2]) * int(sub[4]))
        num += n * power_norm_factor(Mp, Mq)
        den += n
    return num / den


# ======================================================================================
# O4 / O7  centred subgrid DFT pair, each with a factor 1/L^2   (Eq. 7-8 :107-117; R1, R2)
# ======================================================================================
def _dft_matrix(L, sign):
    i = np.arange(L, dtype=np.float64) - L // 2
    return np.exp(sign * 2j * np.pi * np.outer(i, i) / L)


def subgrid_fft(Sp):
    """Shat[gy,gx] = L^-2 sum_{y,x} S'[y,x] exp(-2 pi i[(gy-L/2)(y-L/2)+(gx-L/2)(x-L/2)]/L)."""
    L = Sp.shape[0]
    F = _dft_matrix(L, -1.0)
    return np.einsum("gy,yxp,hx->ghp", F, Sp, F, optimize=True) / (L * L)


def subgrid_ifft(patch):
    """S[y,x] = L^-2 sum_{gy,gx} patch[gy,gx] exp(+2 pi i[...]/L)   (the 1/L^2 is R2)."""
    L = patch.shape[0]
    F = _dft_matrix(L, +1.0)
    return np.einsum("yg,ghp,xh->yxp", F, patch, F, optimize=True) / (L * L)


# ======================================================================================
# O5 / O6  adder and splitter   (Eq. 6 :102, :158, :169)
# ======================================================================================
def adder(grid, Shat, sub, wl_min):
    """grid[wl - wl_min, pol, y0+gy, x0+gx] += Shat[gy, gx, pol]."""
    L = Shat.shape[0]
    x0, y0, wl = int(sub[5]), int(sub[6]), int(sub[7])
    grid[wl - wl_min, :, y0:y0 + L, x0:x0 + L] += np.moveaxis(Shat, 2, 0)


def splitter(grid, sub, L, wl_min):
    """patch[gy, gx, pol] = grid[wl - wl_min, pol, y0+gy, x0+gx]."""
    x0, y0, wl = int(sub[5]), int(sub[6]), int(sub[7])
    return np.moveaxis(np.asarray(grid[wl - wl_min, :, y0:y0 + L, x0:x0 + L], np.complex128), 0, 2)


# ======================================================================================
# O9  degridder: V_k = sum_{y,x} S'[y,x] exp(-2 pi i phi)     (Eq. 13 :171-174)
# ======================================================================================
def degridder_subgrid(par, sub, uvw_m, freqs, Sp):
    """Sp [L,L,4] (after taper and A-term) -> complex128 [nt, nc, 4]."""
    b, t0, nt, c0, nc = (int(v) for v in sub[:5])
    _, du, dv, dw = _subgrid_relative_uvw(par, sub, uvw_m, freqs)
    E = np.exp(-2j * np.pi * _phase(par, du, dv, dw))    # one sum over the pixels, as Eq. 13 is written
    out = np.einsum("kyx,yxp->kp", E, Sp)
    if subgrid_conjugated(par, sub, uvw_m):
        out = dagger(out)                                # predicted V(-u,-v,-w) of (q,p) -> V(u,v,w) of (p,q)
    return out.reshape(nt, nc, 4)


# ======================================================================================
# per-subgrid composites (what the parity tests compare stage by stage)
# ======================================================================================
def grid_subgrid(par, sub, uvw_m, freqs, vis, baselines, aterms, taper):
    """Steps O2-O4 for one subgrid -> (S' after A-term+taper [L,L,4], Shat after FFT [L,L,4])."""
    S = gridder_subgrid(par, sub, uvw_m, freqs, vis)
    Mp, Mq = subgrid_jones(par, sub, baselines, aterms, uvw_m)
    Sp = aterm_taper(S, Mp, Mq, taper, power_norm=par.power_norm)
    return Sp, subgrid_fft(Sp)


def degrid_subgrid(par, sub, uvw_m, freqs, grid, wl_min, baselines, aterms, taper):
    """Steps O6-O9 for one subgrid -> (S' [L,L,4] fed to the degridder, vis [nt,nc,4]).

    R4: the taper multiplies in both directions (Eq. 13's '/T' is read as the caller's
    image-level correction); R5: the same sandwich M_p X M_q^H with the maps given.
    """
    L = par.subgrid_size
    patch = splitter(grid, sub, L, wl_min)
    S = subgrid_ifft(patch)
    Mp, Mq = subgrid_jones(par, sub, baselines, aterms, uvw_m)
    Sp = aterm_taper(S, Mp, Mq, taper)                   # prediction is not power-normalised (R22)
    return Sp, degridder_subgrid(par, sub, uvw_m, freqs, Sp)


# ======================================================================================
# whole path  (§2.5 :152-174)
# ======================================================================================
def layer_range(subgrids):
    if len(subgrids) == 0:
        return 0, 1
    wl_min = int(subgrids[:, 7].min())
    return wl_min, int(subgrids[:, 7].max()) - wl_min + 1


def grid(par, subgrids, uvw_m, freqs, vis, baselines, aterms, taper, out=None):
    """Imaging direction, steps 2.i-2.iii of PAPER.md:155-158 -> grid [W,4,Ng,Ng] complex128."""
    wl_min, W = layer_range(subgrids)
    Ng = par.grid_size
    G = np.zeros((W, 4, Ng, Ng), np.complex128) if out is None else out
    for sub in subgrids:
        _, Shat = grid_subgrid(par, sub, uvw_m, freqs, vis, baselines, aterms, taper)
        adder(G, Shat, sub, wl_min)
    return G


def degrid(par, subgrids, uvw_m, freqs, grid_, baselines, aterms, taper, out=None):
    """Prediction direction, steps 3.i-3.iii of PAPER.md:168-174 -> vis [n_rows,n_chan,4].

    Visibilities not covered by a subgrid (dropped by the planner) are left untouched.
    """
    wl_min, _ = layer_range(subgrids)
    n_rows = uvw_m.shape[0]
    V = np.zeros((n_rows, par.n_chan, 4), np.complex128) if out is None else out
    for sub in subgrids:
        b, t0, nt, c0, nc = (int(v) for v in sub[:5])
        _, v = degrid_subgrid(par, sub, uvw_m, freqs, grid_, wl_min, baselines, aterms, taper)
        r0 = b * par.n_times + t0
        V[r0:r0 + nt, c0:c0 + nc, :] = v
    return V


# ======================================================================================
# closure outside the hot path (w-stacking, Eq. 11 :145-148 and Eq. 12 :166),
# used only to pin the oracle against the measurement equation (P1, P2, P5)
# ======================================================================================
def image_at_pixels(par, G, wl_min, jy, jx):
    """Dirty image BEFORE the division by T_full, at full-image pixels (jy[i], jx[k]) (outer
    product of the two index lists) -> complex128 [len(jy), len(jx), 4].

    I[j] = sum_layers exp(+2 pi i w0 n'(l_j,m_j)) sum_g grid[layer][g] exp(+2 pi i (g-Ng/2)(j-Ng/2)/Ng)
    """
    Ng, S = par.grid_size, par.image_size
    g = np.arange(Ng, dtype=np.float64) - Ng // 2
    jy = np.asarray(jy); jx = np.asarray(jx)
    Ey = np.exp(2j * np.pi * np.outer(jy - Ng // 2, g) / Ng)      # [jy, gy]
    Ex = np.exp(2j * np.pi * np.outer(jx - Ng // 2, g) / Ng)      # [jx, gx]
    l = (jx - Ng // 2) * S / Ng
    m = (jy - Ng // 2) * S / Ng
    n1 = nprime(l[None, :], m[:, None])
    out = np.zeros((jy.size, jx.size, 4), np.complex128)
    for k in range(G.shape[0]):
        w0 = (wl_min + k + 0.5) * par.w_step if par.w_step > 0 else 0.0
        img = np.einsum("ag,pgh,bh->abp", Ey, G[k], Ex, optimize=True)
        out += np.exp(2j * np.pi * w0 * n1)[:, :, None] * img
    return out


def model_to_grid(par, model, wl_min, W):
    """Inverse w-stacking of a model image (already divided by T_full by the caller, R4):
    grid[layer][g] = sum_j model[j] exp(-2 pi i w0 n'_j) exp(-2 pi i (g-Ng/2)(j-Ng/2)/Ng).
    model: complex [4, Ng, Ng] -> complex128 [W, 4, Ng, Ng]."""
    Ng, S = par.grid_size, par.image_size
    j = np.arange(Ng, dtype=np.float64) - Ng // 2
    E = np.exp(-2j * np.pi * np.outer(j, j) / Ng)                  # [g, j]
    l = j * S / Ng
    n1 = nprime(l[None, :], l[:, None])
    G = np.zeros((W, 4, Ng, Ng), np.complex128)
    for k in range(W):
        w0 = (wl_min + k + 0.5) * par.w_step if par.w_step > 0 else 0.0
        scr = np.exp(-2j * np.pi * w0 * n1)
        G[k] = np.einsum("ga,pab,hb->pgh", E, np.asarray(model, np.complex128) * scr[None], E, optimize=True)
    return G
