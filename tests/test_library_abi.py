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
        idg.plan_from_config(synth.scaled(cfg, subgrid_size=48), obs.uvw, obs.freqs, obs.baselines)
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
