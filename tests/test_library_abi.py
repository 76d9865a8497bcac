"""CPU-side checks of the C-ABI library: it loads, exports every symbol include/idg_b200.h
declares, validates its arguments, and its host planner is bit-identical to the oracle's
(SURVEY.md §8(c) "bit-exactly for the subgrid plan and indexing").  No device calls here."""
import os
import re

import numpy as np
import pytest

import synth
from oracle import idg_oracle as orc
from tests.util import oracle_params

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def test_header_symbols_exported(idg):
    header = open(os.path.join(ROOT, "include", "idg_b200.h")).read()
    declared = set(re.findall(r"IDG_API\s+[\w\s\*]+?\b(idg_\w+)\s*\(", header))
    assert declared, "no declarations found in the header"
    assert declared == set(idg.SYMBOLS)
    lib = idg.load_library()
    for name in declared:
        assert hasattr(lib, name), name
    assert "sm_100a" in idg.version()


def _plan(idg, cfg, obs, **kw):
    return idg.plan_from_config(cfg, obs.uvw, obs.freqs, obs.baselines, **kw)


CASES = [
    ("cfg1", lambda: synth.get_config(1)),
    ("cfg2-16st", lambda: synth.scaled(synth.get_config(2), n_stations=16)),
    ("cfg3-12st-layers", lambda: synth.scaled(synth.get_config(3), n_stations=12, n_times=24, n_chan=96)),
    ("cfg4-24st", lambda: synth.scaled(synth.get_config(4), n_stations=24, n_times=8)),
    ("ragged", lambda: synth.scaled(synth.get_config(1), n_stations=7, n_times=13, n_chan=5, aterm_period=3)),
    ("L128", lambda: synth.scaled(synth.get_config(2), n_stations=10, n_times=16, subgrid_size=128, padding=24)),
    ("drops", lambda: synth.scaled(synth.get_config(2), n_stations=12, n_times=8, grid_size=512, cell_arcsec=300.0)),
    ("L48", lambda: synth.scaled(synth.get_config(1), subgrid_size=48, padding=10)),
    ("L160", lambda: synth.scaled(synth.get_config(2), n_stations=8, n_times=8, subgrid_size=160, padding=24)),
]


@pytest.mark.parametrize("name,make", CASES, ids=[c[0] for c in CASES])
def test_plan_bit_exact_vs_oracle(idg, name, make):
    cfg = make()
    obs = synth.make_observation(cfg, vis=None, with_aterms=False)
    sub_o, dropped_o = orc.plan(oracle_params(cfg), obs.uvw, obs.freqs, cfg.n_baselines)
    plan = _plan(idg, cfg, obs)
    cnt = plan.counts()
    sub_c = plan.export()
    assert sub_c.dtype == np.int32 and sub_c.shape == sub_o.shape
    assert np.array_equal(sub_c, sub_o)
    assert cnt.n_subgrids == len(sub_o)
    assert cnt.n_vis_dropped == dropped_o
    assert cnt.n_vis_planned == int((sub_o[:, 2].astype(np.int64) * sub_o[:, 4]).sum())
    assert cnt.n_vis_planned + cnt.n_vis_dropped == cfg.n_vis
    wl_min, W = orc.layer_range(sub_o)
    assert (cnt.wl_min, cnt.n_wlayers) == (wl_min, W)
    if name == "drops":
        assert dropped_o > 0, "case must exercise dropped visibilities"
    if name == "cfg3-12st-layers":
        assert W > 2, "case must exercise several w-layers"


@pytest.mark.parametrize("name,make", [CASES[2], CASES[6]], ids=["cfg3-12st-layers", "drops"])
def test_plan_positive_w_bit_exact_vs_oracle(idg, name, make):
    """PAPER.md:178 (fn 4), R21: with positive_w the C++ planner and the oracle's still agree element for element,
    only layers wl >= 0 remain, every visibility stays planned, and rows with w < 0 sit in subgrids of their own."""
    import dataclasses
    cfg = make()
    obs = synth.make_observation(cfg, vis=None, with_aterms=False)
    par = dataclasses.replace(oracle_params(cfg), positive_w=True)
    sub_o, dropped_o = orc.plan(par, obs.uvw, obs.freqs, cfg.n_baselines)
    plan = _plan(idg, cfg, obs, positive_w=True)
    cnt = plan.counts()
    assert np.array_equal(plan.export(), sub_o) and cnt.n_vis_dropped == dropped_o
    assert cnt.wl_min >= 0
    assert cnt.n_vis_planned + cnt.n_vis_dropped == cfg.n_vis
    if name == "cfg3-12st-layers":
        signed = _plan(idg, cfg, obs).counts()
        assert signed.wl_min < 0 and cnt.n_wlayers < signed.n_wlayers, "conjugation must remove the negative layers"
        w = obs.uvw[:, 2].reshape(cfg.n_baselines, cfg.n_times)
        for b, t0, nt in sub_o[:, :3]:
            sg = np.sign(w[b, t0:t0 + nt])
            assert np.all(sg == sg[0]) or np.all(w[b, t0:t0 + nt] >= 0) or np.all(w[b, t0:t0 + nt] < 0)


def test_config3_full_size_layers_halve_with_positive_w(idg):
    """BASELINE.json configs[2] at full size (host planner only): 10 signed w-layers of 50 lambda become 5 with
    positive_w (PAPER.md:178 fn 4: the conjugation 'halves the number of w-layers'), with the same subgrid count and
    every visibility still planned."""
    cfg = synth.get_config(3)
    obs = synth.make_observation(cfg, vis=None, with_aterms=False)
    signed = _plan(idg, cfg, obs).counts()
    pos = _plan(idg, cfg, obs, positive_w=True).counts()
    assert (signed.n_wlayers, signed.wl_min) == (10, -5) and (pos.n_wlayers, pos.wl_min) == (5, 0)
    assert signed.n_vis_planned == pos.n_vis_planned == cfg.n_vis and pos.n_vis_dropped == 0
    assert signed.n_subgrids == pos.n_subgrids == 517794


def test_kernel_choice_per_subgrid(idg):
    """PAPER.md:247 (fn 7): under AUTO the gridder's subgrids go to the tensor-core kernel
    where at least 65 % of the slots of their 16-channel chunks are filled, to the SIMT kernel otherwise; every
    subgrid takes the tensor-core degridder; forced variants take everything; batches do not change the split."""
    cfg = synth.scaled(synth.get_config(3), n_stations=6, n_times=8)         # 1 ... 384 channels per subgrid
    obs = synth.make_observation(cfg, vis=None, with_aterms=False)
    plan = _plan(idg, cfg, obs)
    sub = plan.export()
    nc = sub[:, 4].astype(np.int64)
    want_tc = int((100 * nc >= 65 * ((nc + 15) // 16 * 16)).sum())
    assert 0 < want_tc < len(sub), "case must mix both kinds"
    assert plan.kernel_split(idg.IDG_GRID) == (want_tc, len(sub) - want_tc)
    assert plan.kernel_split(idg.IDG_DEGRID) == (len(sub), 0)
    assert _plan(idg, cfg, obs, max_batch_subgrids=7).kernel_split(idg.IDG_GRID) == (want_tc, len(sub) - want_tc)
    assert _plan(idg, cfg, obs, gridder_variant=idg.VARIANT_SIMT).kernel_split(idg.IDG_GRID) == (0, len(sub))
    assert _plan(idg, cfg, obs, gridder_variant=idg.VARIANT_TENSOR).kernel_split(idg.IDG_GRID) == (len(sub), 0)
    # config 1: 4 channels per row -> all SIMT; config 2: 32 -> all tensor-core
    for cid, all_tc in ((1, False), (2, True)):
        c = synth.scaled(synth.get_config(cid), n_stations=8)
        o = synth.make_observation(c, vis=None, with_aterms=False)
        nt, ns = _plan(idg, c, o).kernel_split(idg.IDG_GRID)
        assert (ns == 0) if all_tc else (nt == 0)
    # a shape whose tables the tensor-core gridder cannot hold (1300 channels > 1264) runs the SIMT kernel whatever
    # was asked for, and the split says so (what launches is what is reported)
    c = synth.scaled(synth.get_config(1), n_stations=3, n_times=4, n_chan=1300, chan_width_hz=150.0)
    o = synth.make_observation(c, vis=None, with_aterms=False)
    for v in (idg.VARIANT_AUTO, idg.VARIANT_TENSOR):
        p = _plan(idg, c, o, gridder_variant=v)
        assert p.kernel_split(idg.IDG_GRID) == (0, p.counts().n_subgrids)


def test_workspace_follows_batch_capacity(idg):
    cfg = synth.get_config(1)
    obs = synth.make_observation(cfg, vis=None, with_aterms=False)
    n = _plan(idg, cfg, obs).counts().n_subgrids
    L = cfg.subgrid_size
    assert _plan(idg, cfg, obs).workspace_bytes() == n * 4 * L * L * 8
    assert _plan(idg, cfg, obs, max_batch_subgrids=5).workspace_bytes() == 5 * 4 * L * L * 8


def test_argument_validation(idg):
    cfg = synth.get_config(1)
    obs = synth.make_observation(cfg, vis=None, with_aterms=False)
    with pytest.raises(idg.IdgError, match="ascending"):
        idg.plan_from_config(cfg, obs.uvw, obs.freqs[::-1].copy(), obs.baselines)
    bad = obs.baselines.copy()
    bad[0, 1] = cfg.n_stations
    with pytest.raises(idg.IdgError, match="station index"):
        idg.plan_from_config(cfg, obs.uvw, obs.freqs, bad)
    with pytest.raises(idg.IdgError, match="code -2"):
        idg.plan_from_config(synth.scaled(cfg, subgrid_size=40), obs.uvw, obs.freqs, obs.baselines)
    with pytest.raises(idg.IdgError, match="kernel variant"):
        idg.plan_from_config(cfg, obs.uvw, obs.freqs, obs.baselines, gridder_variant=7)
    with pytest.raises(idg.IdgError):
        idg.plan_from_config(synth.scaled(cfg, padding=40), obs.uvw, obs.freqs, obs.baselines)


def test_empty_plan(idg):
    """No baselines: zero subgrids, one (empty) layer, zero workspace."""
    cfg = synth.scaled(synth.get_config(1), n_stations=1)
    plan = idg.Plan(grid_size=cfg.grid_size, subgrid_size=cfg.subgrid_size, padding=cfg.padding,
                    cell_size=cfg.cell_size, w_step=0.0, n_stations=1, n_times=cfg.n_times, n_chan=cfg.n_chan,
                    aterm_period=cfg.aterm_period, uvw_m=np.zeros((0, 3)), freqs=synth.channel_freqs(cfg),
                    baselines=np.zeros((0, 2), np.int32))
    cnt = plan.counts()
    assert (cnt.n_subgrids, cnt.n_wlayers, cnt.n_vis_planned, cnt.n_vis_dropped) == (0, 1, 0, 0)
    assert plan.export().shape == (0, 8)
    # the host-buffer entry points must not index per-layer tables that were never built (round-1 advisor finding)
    assert plan.host_traffic_bytes(idg.IDG_GRID) == (0, 0) and plan.host_traffic_bytes(idg.IDG_DEGRID) == (0, 0)


def test_binding_checks_dtype_and_size(idg):
    """The C ABI sees only pointers: the binding refuses arrays of the wrong dtype or element count."""
    import torch
    cfg = synth.get_config(1)
    obs = synth.make_observation(cfg, vis=None, with_aterms=False)
    plan = _plan(idg, cfg, obs)
    L = cfg.subgrid_size
    ok_vis = torch.zeros((cfg.n_rows, cfg.n_chan, 4), dtype=torch.complex64)
    at = torch.zeros((cfg.n_stations, cfg.n_intervals, L, L, 2, 2), dtype=torch.complex64)
    tp = torch.zeros((L, L), dtype=torch.float32)
    grid = torch.zeros((1, 4, cfg.grid_size, cfg.grid_size), dtype=torch.complex64)
    arena = type("FakeCuda", (), {"is_cuda": True})()       # only the checks before any device work are reached
    with pytest.raises(ValueError, match="dtype float32"):
        idg.grid_host(plan, ok_vis.real.contiguous().repeat(1, 1, 1), at, tp, grid, arena)
    with pytest.raises(ValueError, match="elements, expected"):
        idg.grid_host(plan, ok_vis[:-1], at, tp, grid, arena)
    with pytest.raises(ValueError, match="aterms"):
        idg.grid_host(plan, ok_vis, at[:, :1], tp, grid, arena)
    with pytest.raises(ValueError, match="grid"):
        idg.degrid_host(plan, grid[:, :2], at, tp, ok_vis, arena)


def test_device_calls_fail_loudly_without_cuda_tensors(idg):
    """The product path has no CPU fallback: host tensors are rejected before any work."""
    import torch
    cfg = synth.get_config(1)
    obs = synth.make_observation(cfg, vis=None, with_aterms=False)
    plan = _plan(idg, cfg, obs)
    t = torch.zeros(4)
    with pytest.raises(idg.IdgError, match="no CPU fallback"):
        idg.grid(plan, t, t, t, t, t)
    with pytest.raises(idg.IdgError, match="no CPU fallback"):
        idg.subgrid_fft(32, torch.zeros(32, 32, dtype=torch.complex64), +1)
