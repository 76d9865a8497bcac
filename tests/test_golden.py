"""Stored expected values under tests/golden/ (written by tests/golden/make_golden.py from oracle/ only)."""
import os

import numpy as np

import synth
from oracle import idg_oracle as orc
from tests.util import oracle_params

GOLD = os.path.join(os.path.dirname(os.path.abspath(__file__)), "golden")


def test_plan_config1_oracle_and_library_match_golden(idg):
    """The subgrid table of config 1: oracle planner, C++ planner and the stored table agree bit for bit."""
    gold = np.loadtxt(os.path.join(GOLD, "plan_config1.txt"), dtype=np.int64).astype(np.int32)
    cfg = synth.get_config(1)
    obs = synth.make_observation(cfg, vis=None, with_aterms=False)
    sub, dropped = orc.plan(oracle_params(cfg), obs.uvw, obs.freqs, cfg.n_baselines)
    assert dropped == 0 and np.array_equal(sub, gold)
    plan = idg.plan_from_config(cfg, obs.uvw, obs.freqs, obs.baselines)
    assert np.array_equal(plan.export(), gold)
    # every visibility in exactly one subgrid
    assert int((gold[:, 2].astype(np.int64) * gold[:, 4]).sum()) == cfg.n_vis


def test_gridding_kernel_golden_is_the_closed_form():
    """kernel_L32_P8.txt against K(d) = L^-1 sum_i t[i] exp(2 pi i d (i - L/2) / L) summed term by term here
    (IDG 'effects the same outcome' as convolutional gridding with the taper's transform)."""
    tab = np.loadtxt(os.path.join(GOLD, "kernel_L32_P8.txt"))
    L, P = 32, 8
    t = synth.kaiser_bessel_1d(L, P)
    for d, re, im in tab:
        k = sum(t[i] * np.exp(2j * np.pi * d * (i - L // 2) / L) for i in range(L)) / L
        assert abs(k - (re + 1j * im)) < 1e-14
    # a visibility on a pixel: the deposited values sum to T(0) = 1 (R2)
    on_pixel = tab[np.isclose(tab[:, 0] % 1.0, 0.0)]
    full = sum(t[i] * np.exp(2j * np.pi * np.arange(-L // 2, L // 2)[:, None] * (i - L // 2) / L)
               for i in range(L)) / L
    assert abs(full.sum() - 1.0) < 1e-13 and len(on_pixel) == 9
