"""bench.py -- the IDG hot path (grid + degrid) timed on B200, with its roofline and the oracle beside it.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--config C] [--impl ours|reference]

A "step" is one pass of the whole hot path over one seeded synthetic observation: idg_grid
(gridder -> A-term/taper -> subgrid FFT -> adder) followed by idg_degrid (splitter -> inverse FFT
-> taper/A-term -> degridder) over every visibility of the workload.  `value` = visibilities that
went through BOTH directions per second (n_vis / step time); the per-direction rates are in
`grid_vis_per_s` / `degrid_vis_per_s`.  Workload: BASELINE.json configs[1] (MWA Phase I-like, 128
stations, L = 64), the one the 60 % roofline target is quoted on.  Multi-GPU: the path is specified
for one GPU (replicas only) -- with --gpus N every rank runs the same
workload on its own GPU, no collective on the data path, value = N * n_vis / max-over-ranks time.

Prints ONE JSON line on rank 0.  `--impl reference` times the fp64 numpy oracle (oracle/) on the
host cores on a bounded sample of the same workload and prints the same line shape.
"""
from __future__ import annotations

import argparse
import csv
import json
import os
import subprocess
import sys
import tempfile
import time

import numpy as np

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

import synth  # noqa: E402

METRIC = "gridded+degridded visibilities/s (grid then degrid of every visibility, 4 pols each)"
UNIT = "vis/s"
N_SM = 148
FP32_LANES_PER_SM = 128          # FFMA lanes per SM per clock (micro-benchmarked)
FP32_OPS_PER_PAIR = 18           # 16 FFMA (2x2 complex MAC) + 1 phase FFMA + 1 range-reduction FMUL
MUFU_PER_PAIR = 2


def replicas_aggregate(local_seconds, units_per_rank, world, group=None):
    """Whole-job figures of N independent replicas (the path does not shard in this
    build, so every rank runs the same workload with no data-path collective).  The job's time is the MAX
    over ranks of the device-timed region, and the job processed world x units_per_rank units in it.
    Returns (seconds, units per second).  Works on any backend (the CPU tests run it over gloo)."""
    import torch
    import torch.distributed as dist
    t = torch.tensor([float(local_seconds)], dtype=torch.float64)
    if world > 1:
        if dist.get_backend(group) == "nccl":
            t = t.cuda()
        dist.all_reduce(t, op=dist.ReduceOp.MAX, group=group)
    seconds = float(t.item())
    return seconds, world * units_per_rank / seconds


def load_peaks():
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(p):
        with open(p) as f:
            d = json.load(f)
        return dict(hbm_gbs=float(d["hbm_gbs"]), sm_max_mhz=float(d["sm_max_mhz"]), source="measured")
    return dict(hbm_gbs=6650.0, sm_max_mhz=1965.0, source="fallback")


# ---------------------------------------------------------------------------------------------
# oracle on the host cores (cpu_baseline leg and --impl reference): a bounded sample of subgrids
# ---------------------------------------------------------------------------------------------
_W = {}


def _w_grid(i):
    from oracle import idg_oracle as orc
    w = _W
    _, shat = orc.grid_subgrid(w["par"], w["sub"][i], w["uvw"], w["freqs"], w["vis"], w["bl"], w["aterms"], w["taper"])
    return i, shat


def _w_degrid(i):
    from oracle import idg_oracle as orc
    w = _W
    _, v = orc.degrid_subgrid(w["par"], w["sub"][i], w["uvw"], w["freqs"], w["grid"], w["wl_min"], w["bl"],
                              w["aterms"], w["taper"])
    return i, complex(v.sum())


def oracle_params(cfg):
    from oracle import idg_oracle as orc
    return orc.OracleParams(grid_size=cfg.grid_size, subgrid_size=cfg.subgrid_size, padding=cfg.padding,
                            cell_size=cfg.cell_size, w_step=cfg.w_step, n_times=cfg.n_times, n_chan=cfg.n_chan,
                            aterm_period=cfg.aterm_period, comfort=cfg.comfort)


def oracle_sample(cfg, obs, n_subgrids, seed):
    """A seeded sample of the workload for the oracle: random baselines, planned by the ORACLE's own
    planner (O1), their rows renumbered 0..n-1 so that only those baselines' uvw rows and
    visibilities have to exist on the host.  Input marshalling only; returns a dict for
    oracle_sample_run."""
    from oracle import idg_oracle as orc
    par = oracle_params(cfg)
    rng = np.random.default_rng(seed)
    order = rng.permutation(cfg.n_baselines)
    per_bl = max(1, cfg.n_intervals)                      # at least one subgrid per interval
    n_bl = int(min(cfg.n_baselines, max(1, -(-n_subgrids // per_bl))))
    bls = np.sort(order[:n_bl])
    rows = (bls[:, None].astype(np.int64) * cfg.n_times + np.arange(cfg.n_times)[None, :]).reshape(-1)
    uvw = obs.uvw[rows]
    sub, _ = orc.plan(par, uvw, obs.freqs, n_bl)          # baselines 0..n_bl-1 of the compact table
    if len(sub) > n_subgrids:
        keep = np.sort(rng.choice(len(sub), n_subgrids, replace=False))
        sub = sub[keep]
    vis = synth.source_visibilities(uvw, obs.freqs, obs.sources)
    return dict(par=par, sub=sub, uvw=uvw, freqs=obs.freqs, vis=vis, bl=obs.baselines[bls], aterms=obs.aterms,
                taper=obs.taper)


def oracle_sample_run(cfg, sample, workers):
    """Times the oracle (as it stands) over the sampled subgrids: O2-O5 then O6-O9, in a fork pool
    of `workers` processes.  Returns (n_vis_sampled, seconds)."""
    import multiprocessing as mp
    from oracle import idg_oracle as orc
    sub = sample["sub"]
    wl_min, W = orc.layer_range(sub)
    Ng = cfg.grid_size
    _W.update(sample)
    _W["wl_min"] = wl_min
    ctx = mp.get_context("fork")
    idx = list(range(len(sub)))
    t0 = time.perf_counter()
    G = np.zeros((W, 4, Ng, Ng), np.complex64)          # lazily allocated; only sampled patches are touched
    with ctx.Pool(workers, initializer=_pool_init) as pool:
        for i, shat in pool.imap_unordered(_w_grid, idx):
            orc.adder(G, shat, sub[i], wl_min)
    _W["grid"] = G
    with ctx.Pool(workers, initializer=_pool_init) as pool:
        chk = sum(v for _, v in pool.imap_unordered(_w_degrid, idx))
    dt = time.perf_counter() - t0
    _W.clear()
    assert np.isfinite(chk.real)
    n_vis = int((sub[:, 2].astype(np.int64) * sub[:, 4]).sum())
    return n_vis, dt


def host_workers():
    try:
        return len(os.sched_getaffinity(0))
    except AttributeError:
        return os.cpu_count() or 1



def _pool_init():
    try:
        from threadpoolctl import threadpool_limits
        _W["_limit"] = threadpool_limits(1)               # one BLAS thread per worker: the pool owns the cores
    except Exception:
        pass


def calibrated_oracle(cfg, obs, target_s, seed, workers):
    """Runs the oracle on a small probe sample, then on one sized for about `target_s` seconds of
    wall time.  Returns (vis_per_s, n_vis, seconds, n_subgrids)."""
    probe = oracle_sample(cfg, obs, max(2 * workers, 8), seed)
    n_vis, dt = oracle_sample_run(cfg, probe, workers)
    per_sub = dt / max(len(probe["sub"]), 1)
    n = int(max(len(probe["sub"]), min(target_s / max(per_sub, 1e-6), 4096)))
    if n > len(probe["sub"]) * 1.5:
        sample = oracle_sample(cfg, obs, n, seed + 1)
        n_vis, dt = oracle_sample_run(cfg, sample, workers)
        return n_vis / dt, n_vis, dt, len(sample["sub"])
    return n_vis / dt, n_vis, dt, len(probe["sub"])


def workload_config(cfg):
    return {"workload": f"BASELINE.json configs[{cfg.config_id - 1}] '{cfg.name}': {cfg.n_stations} stations, "
                        f"{cfg.n_baselines} baselines x {cfg.n_times} times x {cfg.n_chan} chan = {cfg.n_vis} vis x 4 pol c64",
            "subgrid_size": cfg.subgrid_size, "padding": cfg.padding, "grid_size": cfg.grid_size,
            "aterm_period": cfg.aterm_period, "w_step": cfg.w_step,
            "l2": "inputs larger than L2 (visibilities + subgrid stack >> 126 MB); no explicit flush"}


def run_reference(args):
    """--impl reference: the fp64 numpy oracle on the host cores, K steps, each a bounded seeded
    sample of the workload (oracle/ is test infrastructure; this is its one timed use)."""
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return 0
    cfg = synth.get_config(args.config)
    obs = synth.make_observation(cfg, vis=None)
    workers = host_workers()
    budget = 150.0                                         # seconds for the whole run
    per_step = max(2.0, budget / max(args.steps + args.warmup, 1))
    probe = oracle_sample(cfg, obs, max(2 * workers, 8), 7)
    _, dt = oracle_sample_run(cfg, probe, workers)        # also serves as the first warm-up
    n_sub = int(max(workers, min(per_step / max(dt / len(probe["sub"]), 1e-6), 2048)))
    for w in range(max(args.warmup - 1, 0)):
        oracle_sample_run(cfg, oracle_sample(cfg, obs, n_sub, 100 + w), workers)
    tot_vis, tot_s, tot_sub = 0, 0.0, 0
    for k in range(args.steps):
        smp = oracle_sample(cfg, obs, n_sub, 200 + k)
        n_vis, dt = oracle_sample_run(cfg, smp, workers)
        tot_vis += n_vis
        tot_s += dt
        tot_sub += len(smp["sub"])
    value = tot_vis / tot_s
    sample = f"{tot_sub // max(args.steps, 1)} seeded random subgrids per step ({tot_vis // max(args.steps, 1)} vis), grid then degrid, fork pool"
    line = {"impl": "reference", "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": args.gpus,
            "steps": args.steps, "warmup": args.warmup, "ms_per_step": 1e3 * tot_s / max(args.steps, 1),
            "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
            "config": workload_config(cfg),
            "cpu_baseline": {"value": value, "unit": UNIT, "cores": workers, "kind": "oracle", "sample": sample},
            "e2e": {"value": value, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
            "gpu_launches": 0}
    print(json.dumps(line))
    return 0


class ClockSampler:
    """nvidia-smi clocks / throttle reasons sampled while the timed region runs (profiling recipe)."""
    FIELDS = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,"
              "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,"
              "clocks_event_reasons.sw_power_cap")

    def __init__(self, index):
        self.f = tempfile.NamedTemporaryFile("w+", suffix=".csv", delete=False)
        self.p = None
        try:
            self.p = subprocess.Popen(["nvidia-smi", "-i", str(index), f"--query-gpu={self.FIELDS}",
                                       "--format=csv,noheader,nounits", "-lms", "50"],
                                      stdout=self.f, stderr=subprocess.DEVNULL)
        except OSError:
            self.p = None

    def stop(self):
        out = {"sm_mhz": None, "sm_max_mhz": None, "reasons": [], "samples": 0}
        if self.p is None:
            return out
        self.p.terminate()
        try:
            self.p.wait(timeout=5)
        except subprocess.TimeoutExpired:
            self.p.kill()
        self.f.flush()
        self.f.seek(0)
        sm, mx, pw, reasons = [], [], [], set()
        names = ("hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap")
        for ln in self.f.read().splitlines():
            parts = [x.strip() for x in ln.split(",")]
            if len(parts) < 7:
                continue
            try:
                sm.append(float(parts[0])); mx.append(float(parts[1])); pw.append(float(parts[2]))
            except ValueError:
                continue
            for nm, val in zip(names, parts[3:7]):
                if val.lower().startswith("active"):
                    reasons.add(nm)
        self.f.close()
        os.unlink(self.f.name)
        if sm:
            out.update(sm_mhz=float(np.median(sm)), sm_max_mhz=float(max(mx)), reasons=sorted(reasons),
                       samples=len(sm), power_w_max=float(max(pw)))
        return out


def kernel_rooflines(cfg, sub, n_wlayers, prof_ms, prof_n, steps, peaks, sm_mhz_obs):
    """Per-kernel achieved rates over the timed region.  ALU kernels (gridder, degridder): algorithmic
    FP32-pipe work = 18 lane-ops per (visibility, pixel) pair, counted as 2 flop each, against
    148 SM x 128 lanes x 2 flop x max SM clock.  HBM kernels (FFT, adder, splitter): algorithmic bytes
    against the measured copy bandwidth.  DESIGN.md "Roofline" derives every figure used here."""
    L, Ng = cfg.subgrid_size, cfg.grid_size
    occ = sub[:, 2].astype(np.int64) * sub[:, 4]
    n_vis = int(occ.sum())
    pairs = float(n_vis) * L * L
    n_sub = len(sub)
    flop = pairs * FP32_OPS_PER_PAIR * 2.0
    peak_tflops = N_SM * FP32_LANES_PER_SM * 2.0 * peaks["sm_max_mhz"] * 1e6 / 1e12
    stack = n_sub * 4.0 * L * L * 8.0
    grid_bytes = n_wlayers * 4.0 * Ng * Ng * 8.0
    aterm_taper = n_sub * (2.0 * L * L * 32.0 + L * L * 4.0)
    alg_bytes = {
        "gridder": n_vis * 32.0 + aterm_taper + stack,
        "degridder": n_vis * 32.0 + aterm_taper + stack,
        "fft": 2.0 * stack, "ifft": 2.0 * stack,
        "adder": stack + 2.0 * grid_bytes,
        "splitter": 2.0 * stack,
    }
    out = {}
    for k, ms in prof_ms.items():
        if prof_n.get(k, 0) == 0:
            continue
        t = ms / 1e3 / steps                                # seconds per step in this kernel
        e = {"ms_per_step": ms / steps, "launches_per_step": prof_n[k] / steps,
             "hbm_gbs": alg_bytes[k] / t / 1e9, "hbm_frac": alg_bytes[k] / t / 1e9 / peaks["hbm_gbs"]}
        if k in ("gridder", "degridder"):
            e.update(bound="alu", tflops=flop / t / 1e12, frac=flop / t / 1e12 / peak_tflops,
                     pairs_per_s=pairs / t,
                     pairs_per_clk_per_sm=(pairs / t) / (N_SM * sm_mhz_obs * 1e6) if sm_mhz_obs else None,
                     frac_at_observed_clock=(flop / t / 1e12) / (peak_tflops * sm_mhz_obs / peaks["sm_max_mhz"])
                     if sm_mhz_obs else None)
        else:
            e.update(bound="hbm", frac=e["hbm_frac"])
        out[k] = e
    return out, peak_tflops, flop, alg_bytes


# What binds the tensor-core direct sums, beside the survey's SIMT roofline (18 FP32-pipe ops per pair, which charges
# the 16 MACs to the FP32 pipe although they run on the tensor pipe, so the gridder can exceed it).  Per (visibility,
# pixel) pair: MUFU operations the shipped kernel issues (rotating gridder: one __sincosf per 8 channels = 0.25;
# degridder: one per pair = 2) and warp instructions ISSUED per pair as ncu counted them in the committed capture
# (profiles/ncu_r03_summary.md: smsp__inst_executed.sum x 32 / pairs).  Peaks per SM clock: 16 SFU lanes
# (MUFU.EX2 measured 16.0, profiles/alu_peaks_r01.md), 4 schedulers x 32 lanes = 128 issued thread-instructions.
CEILING_INPUTS = {"gridder": {"mufu_per_pair": 0.25, "issued_per_pair": 12.4},
                  "degridder": {"mufu_per_pair": 2.0, "issued_per_pair": 14.8}}
SFU_LANES_PER_SM, ISSUE_LANES_PER_SM = 16.0, 128.0


def ceilings(kernel, pairs_per_clk_per_sm):
    """Ceilings of a tensor-core direct-sum kernel in pairs per SM clock, and the fraction of the tightest one that
    is a true bound for it (the SIMT-equivalent FP32 figure is kept as a label, not as a bound)."""
    c = CEILING_INPUTS[kernel]
    sfu = SFU_LANES_PER_SM / c["mufu_per_pair"]
    issue = ISSUE_LANES_PER_SM / c["issued_per_pair"]
    out = {"unit": "pairs/clk/SM", "simt_equivalent_fp32": FP32_LANES_PER_SM / FP32_OPS_PER_PAIR, "sfu": sfu,
           "issue_slots": issue, "mufu_per_pair": c["mufu_per_pair"], "issued_instructions_per_pair": c["issued_per_pair"],
           "source": "profiles/ncu_r03_summary.md (instructions per pair), profiles/alu_peaks_r01.md (pipe widths)",
           "binding": "sfu" if sfu < issue else "issue_slots"}
    if pairs_per_clk_per_sm:
        out["achieved"] = pairs_per_clk_per_sm
        out["frac_of_binding"] = pairs_per_clk_per_sm / min(sfu, issue)
    return out


VARIANTS = {"auto": 0, "simt": 1, "tensor": 2, "fp64": 3}      # IDG_VARIANT_* of include/idg_b200.h
OPERANDS = ("direct sums on tcgen05: gridder fp16 head + fp16 remainder of (cos, sin) and of the visibilities (one "
            "power-of-two scale per segment), degridder tf32 head + tf32 remainder; fp32 accumulation in tensor memory, "
            "drained into fp32 registers every 12 chunks; phase, sin/cos, A-term sandwich, FFT in fp32, adder sums in "
            "fp64; sparsely filled subgrids take the all-fp32 SIMT kernels (kernel choice per subgrid)")


def device_leg(idg, torch, cfg, plan, sub, cnt, d_vis, d_at, d_tp, steps, warmup, stream, barrier, peaks,
               sampler_index=None, prediction_only=False):
    """Times `steps` passes of the hot path on resident inputs with CUDA events on the launching stream, after
    `warmup` untimed passes.  Returns a dict of whole-step, per-direction and per-kernel figures."""
    Ng = cfg.grid_size
    d_grid = torch.zeros((cnt.n_wlayers, 4, Ng, Ng), dtype=torch.complex64, device=d_vis.device)
    d_out = torch.zeros_like(d_vis)
    ws = torch.empty(max(plan.workspace_bytes(idg.IDG_GRID), plan.workspace_bytes(idg.IDG_DEGRID)),
                     dtype=torch.uint8, device=d_vis.device)
    if prediction_only:                                   # config 5: the grid is an input, made once
        idg.grid(plan, d_vis, d_at, d_tp, d_grid, ws, stream)
    # clocks and throttle reasons are sampled from the warm-up steps on (nvidia-smi takes a moment to start and
    # the timed region of the default run is under a second); the GPU runs the same kernels throughout
    sampler = ClockSampler(sampler_index) if sampler_index is not None else None

    def one(k=None, ev=None):
        if not prediction_only:
            idg.grid(plan, d_vis, d_at, d_tp, d_grid, ws, stream)
        if ev is not None:
            ev[2 * k + 1].record(stream)
        idg.degrid(plan, d_grid, d_at, d_tp, d_out, ws, stream)
        if ev is not None:
            ev[2 * k + 2].record(stream)

    for _ in range(warmup):
        one()
    barrier()
    idg.profile_read()
    idg.profile_enable(True)
    launches0 = idg.launch_count()
    ev = [torch.cuda.Event(enable_timing=True) for _ in range(2 * steps + 1)]
    ev[0].record(stream)
    for k in range(steps):
        one(k, ev)
    barrier()
    launches = idg.launch_count() - launches0
    idg.profile_enable(False)
    prof = idg.profile_read()
    clocks = sampler.stop() if sampler else None
    total_ms = ev[0].elapsed_time(ev[-1])
    grid_ms = sum(ev[2 * k].elapsed_time(ev[2 * k + 1]) for k in range(steps)) / steps
    degrid_ms = sum(ev[2 * k + 1].elapsed_time(ev[2 * k + 2]) for k in range(steps)) / steps
    sm_obs = clocks["sm_mhz"] if clocks else None
    prof_ms = {k: v[0] for k, v in prof.items()}
    prof_n = {k: v[1] for k, v in prof.items()}
    kr, peak_tflops, _, _ = kernel_rooflines(cfg, sub, cnt.n_wlayers, prof_ms, prof_n, steps, peaks, sm_obs)
    n_vis = cnt.n_vis_planned
    out = {"total_ms": total_ms, "ms_per_step": total_ms / steps, "degrid_ms": degrid_ms,
           "degrid_vis_per_s": n_vis / (degrid_ms / 1e3), "kernels": kr, "clocks": clocks, "launches": int(launches),
           "peak_tflops": peak_tflops, "n_subgrids": int(cnt.n_subgrids), "n_vis": int(n_vis),
           "n_wlayers": int(cnt.n_wlayers)}
    if not prediction_only:
        out.update(grid_ms=grid_ms, grid_vis_per_s=n_vis / (grid_ms / 1e3))
    del d_grid, d_out, ws
    return out


def other_config(idg, torch, config_id, dev, stream, barrier, peaks, sampler_index):
    """One warm-up and two timed steps of another BASELINE.json config (1, 3, 4: grid + degrid; config 1 is 56 subgrids
    of 32 visibilities, launch-latency-bound: reported, not tuned for; 5: prediction only, from
    the grid of one imaging pass), visibilities by the counter-based hash recipe generated on the device (the
    values do not affect timing).  The headline `value`, `config` and `roofline` stay config 2's."""
    cfg = synth.get_config(config_id)
    obs = synth.make_observation(cfg, vis=None)
    plan = idg.plan_from_config(cfg, obs.uvw, obs.freqs, obs.baselines)
    sub = plan.export()
    cnt = plan.counts()
    d_vis = synth.hash_visibilities_torch(cfg.n_rows, cfg.n_chan, cfg.seed, dev)
    d_at = torch.from_numpy(obs.aterms).to(dev)
    d_tp = torch.from_numpy(obs.taper).to(dev)
    r = device_leg(idg, torch, cfg, plan, sub, cnt, d_vis, d_at, d_tp, 2, 1, stream, barrier, peaks, sampler_index,
                   prediction_only=(config_id == 5))
    del d_vis, d_at, d_tp, plan
    torch.cuda.empty_cache()
    keep = {k: r[k] for k in ("ms_per_step", "grid_ms", "degrid_ms", "grid_vis_per_s", "degrid_vis_per_s", "n_subgrids",
                              "n_vis", "n_wlayers", "clocks") if k in r}
    keep["workload"] = workload_config(cfg)["workload"]
    keep["steps"], keep["warmup"] = 2, 1
    keep["kernels"] = {k: {"ms_per_step": v["ms_per_step"], "frac": v["frac"], "bound": v["bound"],
                           **({"pairs_per_clk_per_sm": v["pairs_per_clk_per_sm"]} if "pairs_per_clk_per_sm" in v else {})}
                       for k, v in r["kernels"].items()}
    return keep


def run_ours(args):
    import torch
    import torch.distributed as dist

    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    cfg = synth.get_config(args.config)
    peaks = load_peaks()
    obs = synth.make_observation(cfg, vis=None)

    # the oracle beside it: rank 0, N = 1 only, BEFORE CUDA is initialised (it forks a process pool)
    cpu_baseline = None
    if rank == 0 and world == 1 and not args.no_cpu_baseline:
        workers = host_workers()
        v, n_vis_s, dt, n_s = calibrated_oracle(cfg, obs, args.cpu_seconds, 11, workers)
        cpu_baseline = {"value": v, "unit": UNIT, "cores": workers, "kind": "oracle",
                        "sample": f"{n_s} seeded random subgrids ({n_vis_s} vis) of the same workload, grid then "
                                  f"degrid, fork pool, {dt:.1f} s wall"}

    if not torch.cuda.is_available():
        raise RuntimeError("bench.py needs a CUDA device: the IDG path has no CPU fallback")
    from paper_2502_17789_b200 import build as _build
    _build.build()
    import paper_2502_17789_b200 as idg
    torch.cuda.set_device(local)
    dev = torch.device("cuda", local)
    if world > 1:
        dist.init_process_group("nccl", device_id=dev)

    variants = dict(gridder_variant=VARIANTS[args.gridder_variant], degridder_variant=VARIANTS[args.degridder_variant])
    plan = idg.plan_from_config(cfg, obs.uvw, obs.freqs, obs.baselines, max_batch_subgrids=args.max_batch, **variants)
    sub = plan.export()
    cnt = plan.counts()
    Ng = cfg.grid_size
    if cfg.config_id in (3, 4, 5):
        d_vis = synth.hash_visibilities_torch(cfg.n_rows, cfg.n_chan, cfg.seed, dev)
    else:
        d_vis = synth.source_visibilities_torch(obs.uvw, obs.freqs, obs.sources, dev)
    d_at = torch.from_numpy(obs.aterms).to(dev)
    d_tp = torch.from_numpy(obs.taper).to(dev)
    stream = torch.cuda.current_stream()

    def barrier():
        torch.cuda.synchronize()
        if world > 1:
            dist.barrier()
            torch.cuda.synchronize()

    warmup = max(args.warmup, 3)
    prediction_only = cfg.config_id == 5
    leg = device_leg(idg, torch, cfg, plan, sub, cnt, d_vis, d_at, d_tp, args.steps, warmup, stream, barrier, peaks,
                     torch.cuda.current_device() if rank == 0 else None, prediction_only)
    n_vis = cnt.n_vis_planned
    total_s, value = replicas_aggregate(leg["total_ms"] / 1e3, n_vis * args.steps, world)
    ms_per_step = total_s * 1e3 / args.steps

    # end to end through the host-buffer C-ABI calls: pinned host -> device -> pinned host, every step
    e2e = None
    if not args.no_e2e and not prediction_only:
        h_vis = d_vis.cpu().pin_memory()
        h_at = torch.from_numpy(obs.aterms).pin_memory()
        h_tp = torch.from_numpy(obs.taper).pin_memory()
        h_grid = torch.zeros((cnt.n_wlayers, 4, Ng, Ng), dtype=torch.complex64).pin_memory()
        h_out = torch.zeros((cfg.n_rows, cfg.n_chan, 4), dtype=torch.complex64).pin_memory()
        # the host-buffer calls pipeline copies against compute batch by batch: smaller batches overlap more.
        # The device-resident headline keeps the library's default batch; the SAME plan the end-to-end leg uses is
        # also timed device-resident below, so the two legs can be compared on one configuration of the library.
        e2e_plan, same_plan_ms = plan, leg["ms_per_step"]
        if args.e2e_batch and not args.max_batch:
            e2e_plan = idg.plan_from_config(cfg, obs.uvw, obs.freqs, obs.baselines, max_batch_subgrids=args.e2e_batch,
                                            **variants)
            same = device_leg(idg, torch, cfg, e2e_plan, sub, cnt, d_vis, d_at, d_tp, args.steps, 1, stream, barrier, peaks)
            same_plan_ms = same["ms_per_step"]
        torch.cuda.empty_cache()
        arena = torch.empty(max(e2e_plan.host_arena_bytes(idg.IDG_GRID), e2e_plan.host_arena_bytes(idg.IDG_DEGRID)),
                            dtype=torch.uint8, device=dev)
        n_e2e = args.steps
        idg.grid_host(e2e_plan, h_vis, h_at, h_tp, h_grid, arena, stream)        # warm-up
        idg.degrid_host(e2e_plan, h_grid, h_at, h_tp, h_out, arena, stream)
        barrier()
        t0 = time.perf_counter()
        for _ in range(n_e2e):
            idg.grid_host(e2e_plan, h_vis, h_at, h_tp, h_grid, arena, stream)
            idg.degrid_host(e2e_plan, h_grid, h_at, h_tp, h_out, arena, stream)
        torch.cuda.synchronize()
        dt = time.perf_counter() - t0
        dt, e2e_value = replicas_aggregate(dt, n_vis * n_e2e, world)
        # what the two calls move over the bus, from the library (visibility rows and master-grid rows under a
        # subgrid, A-terms, taper; the degrid call uploads visibilities only if the planner left some uncovered)
        up_g, down_g = e2e_plan.host_traffic_bytes(idg.IDG_GRID)
        up_d, down_d = e2e_plan.host_traffic_bytes(idg.IDG_DEGRID)
        h2d, d2h = up_g + up_d, down_g + down_d
        e2e = {"value": e2e_value, "unit": UNIT, "h2d_bytes_per_step": h2d,
               "d2h_bytes_per_step": d2h, "steps": n_e2e, "ms_per_step": 1e3 * dt / n_e2e,
               "api": "idg_grid_host + idg_degrid_host (pinned host buffers; copies inside the calls, "
                      "overlapped with compute per batch on a second stream)",
               "max_batch_subgrids": int(args.max_batch or args.e2e_batch),
               "device_resident_ms_per_step_same_plan": same_plan_ms}
        del arena, h_vis, h_grid, h_out
    del d_vis, d_at, d_tp
    torch.cuda.empty_cache()

    # the other single-GPU workloads of BASELINE.json, briefly (rank 0 of a 1-GPU run only)
    others = None
    if rank == 0 and world == 1 and cfg.config_id == 2 and not args.no_other_configs:
        others = {}
        for c in (1, 3, 4, 5):
            others[str(c)] = other_config(idg, torch, c, dev, stream, barrier, peaks, torch.cuda.current_device())

    if rank != 0:
        if world > 1:
            dist.destroy_process_group()
        return 0
    kr, clocks = leg["kernels"], leg["clocks"]
    cands = [k for k in ("gridder", "degridder") if k in kr]
    dom = max(cands, key=lambda k: kr[k]["ms_per_step"])
    roofline = {"kernel": dom, "bound": "alu", "achieved": kr[dom]["tflops"], "peak": leg["peak_tflops"],
                "unit": "TFLOP/s", "frac": kr[dom]["frac"],
                "traffic": ncu_traffic(dom, cfg, cnt.n_subgrids, kr[dom]["launches_per_step"]),
                "peak_basis": f"{N_SM} SM x {FP32_LANES_PER_SM} FP32 lanes x 2 flop x {peaks['sm_max_mhz']:.0f} MHz "
                              f"(sm_max_mhz {peaks['source']}); work = 18 FP32-pipe ops per (vis,pixel) pair",
                "frac_at_observed_clock": kr[dom]["frac_at_observed_clock"],
                "hbm_frac_of_measured": kr[dom]["hbm_frac"], "hbm_peak_gbs": peaks["hbm_gbs"],
                # `frac` is the survey's SIMT roofline; what actually binds the tensor-core kernels, per kernel:
                "ceilings": {k: ceilings(k, kr[k].get("pairs_per_clk_per_sm")) for k in cands
                             if getattr(args, k + "_variant") in ("auto", "tensor")},
                # every kernel of the headline config (the stored record keeps `roofline`)
                "per_kernel": {k: {"ms_per_step": v["ms_per_step"], "bound": v["bound"], "frac": v["frac"]}
                               for k, v in kr.items()}}
    metric = METRIC if not prediction_only else "degridded (predicted) visibilities/s (4 pols each)"
    line = {"metric": metric, "value": value, "unit": UNIT, "n_gpus": world,
            "steps": args.steps, "warmup": warmup, "ms_per_step": ms_per_step,
            "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f32", "operands": OPERANDS,
            "data": "synthetic", "config": workload_config(cfg), "grid_vis_per_s": leg.get("grid_vis_per_s"),
            "degrid_vis_per_s": leg["degrid_vis_per_s"], "grid_ms": leg.get("grid_ms"), "degrid_ms": leg["degrid_ms"],
            "n_subgrids": int(cnt.n_subgrids), "n_vis": int(n_vis), "roofline": roofline, "kernels": kr,
            "cpu_baseline": cpu_baseline, "e2e": e2e, "gpu_launches": leg["launches"], "clocks": clocks,
            "other_configs": others}
    print(json.dumps(line))
    if world > 1:
        dist.destroy_process_group()
    return 0


def ncu_traffic(kernel, cfg, n_subgrids, launches_per_step):
    """DRAM bytes per launch of the dominant kernel from the committed ncu capture (profiles/), scaled from the
    captured launch to this run's average launch; None when there is no capture for this workload."""
    path = os.path.join(os.path.dirname(os.path.abspath(__file__)), "profiles", "dram_traffic_r03a.csv")
    if cfg.config_id != 2 or not os.path.exists(path) or not launches_per_step:
        return None
    with open(path) as f:
        for row in csv.DictReader(f):
            if row["kernel"] == kernel:
                per_subgrid = (float(row["dram_bytes_read"]) + float(row["dram_bytes_write"])) / float(row["subgrids_in_launch"])
                return per_subgrid * n_subgrids / launches_per_step
    return None


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=5)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--config", type=int, default=2, help="BASELINE.json config id (1-based); default 2 = configs[1]")
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--cpu-seconds", type=float, default=15.0, help="wall-time target of the cpu_baseline leg")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-e2e", action="store_true")
    ap.add_argument("--gridder-variant", default="auto", choices=["auto", "simt", "tensor", "fp64"],
                    help="idg_params.gridder_variant (auto = per subgrid, the library default)")
    ap.add_argument("--degridder-variant", default="auto", choices=["auto", "simt", "tensor", "fp64"])
    ap.add_argument("--no-other-configs", action="store_true",
                    help="skip the brief runs of configs 3, 4 and 5 that follow the config-2 headline")
    ap.add_argument("--e2e-batch", type=int, default=8192,
                    help="subgrids per batch of the plan the end-to-end leg uses (0 = same plan as the device leg)")
    ap.add_argument("--max-batch", type=int, default=0,
                    help="subgrids per batch (0 = the library default: 4 GiB of subgrid stack)")
    args = ap.parse_args()
    if args.impl == "reference":
        return run_reference(args)
    return run_ours(args)


if __name__ == "__main__":
    sys.exit(main())
