"""idg_power_norm_average_static: the entry point for callers that cannot allocate device memory.

Some users of this library must not let it call cudaMalloc: an imager whose own pool took the whole device at
start-up (a raw allocation then fails although the pool has room), or one that prepares the image correction
while gridding batches run on other streams (cudaMalloc / cudaFree synchronise the whole device and stall them).
For them the power-normalisation average (§3.3, R22) exists a second time with its scratch built
into the library (at most L = 96; 4.5 MiB per GPU) and every other buffer passed in by the caller.

The test runs it twice in a row and compares each result with idg_power_norm_average, the allocating path (which
test_gpu_parity.py checks against the oracle): same kernels, same summation order, so the tolerance is that
test's 1e-12 and in fact the bits agree.  The second call uses other A-terms and a poisoned output, so a result
left over in the shared scratch from the first call cannot pass for the second.  The file is named to be
collected last: `pytest -x` stops at the first failure and a failure here must not hide the parity tests.
It passes alone in a fresh process (first use of the scratch on the device) and after the other tests.
"""
import numpy as np
import pytest
import torch

import synth
from tests.util import random_jones

DEV = "cuda:0"


def _plan(idg, **kw):
    cfg = synth.scaled(synth.get_config(2), n_stations=7, n_times=16, grid_size=1024, cell_arcsec=120.0, **kw)
    obs = synth.make_observation(cfg, vis="hash", with_aterms=False)
    return cfg, idg.plan_from_config(cfg, obs.uvw, obs.freqs, obs.baselines, power_norm=True)


def test_power_norm_terms_on_the_host(idg):
    """idg_plan_power_norm_terms needs no GPU: one term per (baseline, interval) that carries planned visibilities,
    weights = visibility counts (they add up to the plan's count), and a capacity that is too small is refused."""
    cfg, plan = _plan(idg)
    sub = plan.export()
    pairs, weights, wsum = idg.plan_power_norm_terms(plan)
    assert pairs.shape == (len(weights), 3) and len(weights) > 0
    assert wsum == weights.sum() == plan.counts().n_vis_planned == int((sub[:, 2] * sub[:, 4]).sum())
    key = {(int(b), int(t0) // cfg.aterm_period) for b, t0 in sub[:, :2]}
    assert len(key) == len(weights)
    assert (pairs[:, 2] >= 0).all() and (pairs[:, 2] < cfg.n_intervals).all() and (pairs[:, :2] < cfg.n_stations).all()
    import ctypes
    lib = idg.load_library()
    small_p, small_w = np.zeros((1, 3), np.int32), np.zeros(1, np.float64)
    rc = lib.idg_plan_power_norm_terms(plan.handle, small_p.ctypes.data, small_w.ctypes.data, 1, None, None)
    assert rc == -3 and b"room for 1" in lib.idg_last_error()
    assert ctypes.c_int(rc).value != 0


@pytest.mark.gpu
def test_static_scratch_matches_allocating_path_twice_in_a_row(idg):
    cfg, plan = _plan(idg)
    L = cfg.subgrid_size
    pairs, weights, wsum = idg.plan_power_norm_terms(plan)
    d_pairs = torch.from_numpy(pairs).to(DEV)
    d_weights = torch.from_numpy(weights).to(DEV)
    rng = np.random.default_rng(31)
    for call in range(2):
        at = random_jones(rng, (cfg.n_stations, cfg.n_intervals, L, L), scale=0.3 + 0.4 * call)
        d_at = torch.from_numpy(at).to(DEV)
        got = torch.full((L, L), float("nan"), dtype=torch.float64, device=DEV)
        idg.power_norm_average_static(d_at, L, cfg.n_intervals, d_pairs, d_weights, wsum, got)
        want = torch.zeros((L, L), dtype=torch.float64, device=DEV)
        idg.power_norm_average(plan, d_at, want)
        torch.cuda.synchronize()
        g, w = got.cpu().numpy(), want.cpu().numpy()
        assert np.isfinite(g).all() and (w > 0).all()
        assert np.abs(g - w).max() <= 1e-12 * np.abs(w).max(), f"call {call}"
        assert np.array_equal(g, w), f"call {call}: same kernels, same order: the bits must agree"
        if call:
            assert not np.array_equal(g, first), "the second call must not return the first call's result"
        first = g


@pytest.mark.gpu
def test_static_scratch_refuses_sizes_beyond_its_maximum(idg):
    """L = 128 does not fit the built-in scratch: a clear error, not a silent overrun; bad arguments likewise."""
    L = 128
    d_at = torch.zeros((2, 1, L, L, 2, 2), dtype=torch.complex64, device=DEV)
    d_pairs = torch.zeros((1, 3), dtype=torch.int32, device=DEV)
    d_w = torch.ones(1, dtype=torch.float64, device=DEV)
    out = torch.zeros((L, L), dtype=torch.float64, device=DEV)
    with pytest.raises(idg.IdgError, match="IDG_STATIC_MAX_SUBGRID_SIZE = 96"):
        idg.power_norm_average_static(d_at, L, 1, d_pairs, d_w, 1.0, out)
    with pytest.raises(idg.IdgError, match="weight_sum > 0"):
        idg.power_norm_average_static(d_at[..., :64, :64, :, :].contiguous(), 64, 1, d_pairs, d_w, 0.0, out[:64, :64].contiguous())
