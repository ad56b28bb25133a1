#!/usr/bin/env python
"""bench.py -- SALT3 batched band-flux throughput on B200 (BASELINE.json metric).

  python bench.py [--gpus N] [--steps K] [--warmup W] [--config 5] [--impl ours|reference]

A step is one `sb_chi2` call (through the C ABI) over the whole workload: every row of the hot
path (rest-frame shift, bicubic interpolation, colour law, band weighting, trapezoid integral, zero
point, chi^2) for every (supernova, sample, observation), writing band flux and chi^2.
`--mode grad` times `sb_bandflux_grad` instead.  Prints ONE JSON line (rank 0).

Default workload: BASELINE.json configs[4] ("survey scale": 100000 SN x 80 obs, NIR grid), the
configuration north_star's throughput target is quoted on; it fits one GPU.  Inputs (8e6
observations x 20 B + 32 MB of output) exceed the 126 MB L2, so no flush is needed; smaller
configs flush L2 between timed steps.  Multi-GPU: one shard of the same size per rank (weak
scaling), no data-path collective.
"""
from __future__ import annotations

import argparse
import json
import os
import subprocess
import sys
import threading
import time

import numpy as np

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

import workloads  # noqa: E402

METRIC = "bandflux_evals_per_sec"
UNIT = "evals/s"

# Flop model of the formulation the kernel executes (FMA = 2, add/mul = 1,
# ex2 = 1; min/max/select/compare/convert/shuffle/address arithmetic = 0).
FLOPS_PER_SAMPLE_FWD = 28  # t FFMA 2, split 3, poly3 6, colour r 2 + d 1 + Horner(4) 8 + cont. 2, ex2 1, E*W 1, acc 2
FLOPS_PER_CELL_FWD = 32    # collapse 8 FFMA = 16, cell coefficients 16
FLOPS_PER_EVAL_FWD = 60    # phase weights, zero point, chi^2 term, butterfly
FLOPS_PER_SAMPLE_GRAD = 46  # + unscaled arg 1, 2 extra poly3 12, f 1, 3 extra accumulators 6 (-1: no pre-scale)
FLOPS_PER_CELL_GRAD = 82    # collapse 16 FFMA + x1 combine = 34, three coefficient sets 48
FLOPS_PER_EVAL_GRAD = 120
# Grouped (node-weight / adjoint) formulation, csrc/sb_hoist.cuh: per band sample of a CHUNK (up to 8
# observations of one (unit, band) share it): colour Horner 8, ex2 1, x W 1, moments 9, steps 2;
# per model cell of a chunk: sample range 9, moments -> node weights 20, x1 1; per node per
# observation: 8 FFMA; per eval: phase weights, zero point, chi^2 term, reduction.
FLOPS_G_SAMPLE, FLOPS_G_CELL, FLOPS_G_NODE_OBS, FLOPS_G_EVAL = 21, 30, 16, 60
# Node-weight ("tiled") formulation, csrc/sb_nw.cuh: the same per-sample and per-cell work once per (unit, band)
# ITEM (all its observations share it); per node per observation 8 FFMA (phase collapse of M0, M1
# with x1 folded into the weights) + 1 FFMA (node weight) = 18.  Only nodes of the item's window count;
# the zero-padded remainder of the 128-node half windows the kernel also multiplies is not counted.
FLOPS_T_NODE_OBS = 18
# Tiled gradient: per sample + CL scaling 1, CL weighting 1, four CL-weighted moments 8 = 31; per cell two
# weight sets 50; per node per observation 21 FFMA = 42 (value, M1-only, d/dt0 rows, four sums).
FLOPS_TG_SAMPLE, FLOPS_TG_CELL, FLOPS_TG_NODE_OBS, FLOPS_TG_EVAL = 31, 50, 42, 120
# SURVEY.md section 8(d) "direct (G = 1)" model, reported beside ours for reference.
SURVEY_SAMPLE, SURVEY_NODE, SURVEY_EVAL = 55, 18, 40
SURVEY_SAMPLE_GRAD, SURVEY_NODE_GRAD, SURVEY_EVAL_GRAD = 77, 36, 100


def geometry_counts(wl):
    """Per observation: in-range band samples n_in and model cells spanned (0 when the phase is
    outside the grid for every sample of the unit -- evaluated at the first sample of each unit)."""
    md, bd = wl.model, wl.bands
    l0, l1 = float(md["wave"][0]), float(md["wave"][-1])
    dl = float(md["wave"][1] - md["wave"][0])
    p0, p1 = float(md["phase"][0]), float(md["phase"][-1])
    n_obs = np.diff(wl.obs_offset)
    z = np.repeat(wl.z.astype(np.float64), n_obs)
    opz = 1.0 + z
    n_in = np.zeros(wl.n_obs_total, dtype=np.int64)
    n_cell = np.zeros(wl.n_obs_total, dtype=np.int64)
    for b in range(wl.n_bands):
        lam = bd["wave"][bd["offset"][b]:bd["offset"][b + 1]]
        sel = np.nonzero(wl.band == b)[0]
        lo = np.searchsorted(lam, l0 * opz[sel], side="left")
        hi = np.searchsorted(lam, l1 * opz[sel], side="right")
        cnt = np.maximum(hi - lo, 0)
        n_in[sel] = cnt
        ok = cnt > 0
        u_first = (lam[np.minimum(lo, len(lam) - 1)] / opz[sel] - l0) / dl
        u_last = (lam[np.maximum(hi - 1, 0)] / opz[sel] - l0) / dl
        n_cell[sel] = np.where(ok, np.floor(u_last) - np.floor(u_first) + 1, 0)
    # phase range (per unit's first sample; configs keep every phase inside the grid)
    t0 = wl.theta["t0"].astype(np.float64).reshape(wl.n_sn, -1)[:, 0]
    p = (wl.time.astype(np.float64) - np.repeat(t0, n_obs)) / opz
    inside = (p >= p0) & (p <= p1)
    return np.where(inside, n_in, 0), np.where(inside, n_cell, 0)


def chunk_share(wl, chunk: int = 8):  # chunk = 0: the whole item is one chunk
    """Per observation: chunks of its (unit, band) item / observations of the item (the fraction of
    the item's shared per-sample and per-cell work that one observation carries)."""
    n_obs = np.diff(wl.obs_offset)
    unit = np.repeat(np.arange(wl.n_sn, dtype=np.int64), n_obs)
    key = unit * wl.n_bands + wl.band.astype(np.int64)
    cnt = np.bincount(key, minlength=wl.n_sn * wl.n_bands)
    c = cnt[key]
    return (np.ceil(c / chunk) if chunk > 0 else 1.0) / c


def flops_per_call(wl, grad: bool, form: str = "direct"):
    n_in, n_cell = geometry_counts(wl)
    ns = wl.n_samples
    s_in, s_cell, n_ev = float(n_in.sum()) * ns, float(n_cell.sum()) * ns, float(wl.n_evals)
    if form == "tiled" and grad:
        share = chunk_share(wl, 0)
        g_in, g_cell = float((n_in * share).sum()) * ns, float((n_cell * share).sum()) * ns
        s_node = float((n_cell + 3 * (n_cell > 0)).sum()) * ns
        ours = g_in * FLOPS_TG_SAMPLE + g_cell * FLOPS_TG_CELL + s_node * FLOPS_TG_NODE_OBS + n_ev * FLOPS_TG_EVAL
        surv = s_in * SURVEY_SAMPLE_GRAD + (s_cell + 3 * n_ev) * SURVEY_NODE_GRAD + n_ev * SURVEY_EVAL_GRAD
        return ours, surv, s_in / max(n_ev, 1.0), s_cell / max(n_ev, 1.0)
    if form in ("grouped", "tiled") and not grad:
        share = chunk_share(wl, 8 if form == "grouped" else 0)
        node_obs = FLOPS_G_NODE_OBS if form == "grouped" else FLOPS_T_NODE_OBS
        g_in, g_cell = float((n_in * share).sum()) * ns, float((n_cell * share).sum()) * ns
        s_node = float((n_cell + 3 * (n_cell > 0)).sum()) * ns
        ours = g_in * FLOPS_G_SAMPLE + g_cell * FLOPS_G_CELL + s_node * node_obs + n_ev * FLOPS_G_EVAL
        surv = s_in * SURVEY_SAMPLE + (s_cell + 3 * n_ev) * SURVEY_NODE + n_ev * SURVEY_EVAL
        return ours, surv, s_in / max(n_ev, 1.0), s_cell / max(n_ev, 1.0)
    if grad:
        ours = s_in * FLOPS_PER_SAMPLE_GRAD + s_cell * FLOPS_PER_CELL_GRAD + n_ev * FLOPS_PER_EVAL_GRAD
        surv = s_in * SURVEY_SAMPLE_GRAD + (s_cell + 3 * n_ev) * SURVEY_NODE_GRAD + n_ev * SURVEY_EVAL_GRAD
    else:
        ours = s_in * FLOPS_PER_SAMPLE_FWD + s_cell * FLOPS_PER_CELL_FWD + n_ev * FLOPS_PER_EVAL_FWD
        surv = s_in * SURVEY_SAMPLE + (s_cell + 3 * n_ev) * SURVEY_NODE + n_ev * SURVEY_EVAL
    return ours, surv, s_in / max(n_ev, 1.0), s_cell / max(n_ev, 1.0)


class ClockSampler:
    """nvidia-smi clocks / throttle reasons sampled every 20 ms.  Started before the warm-up (the tool needs
    tens of milliseconds to come up); stop(t0, t1) keeps the samples that arrived inside the timed region."""

    Q = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,"
         "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,"
         "clocks_event_reasons.sw_power_cap")

    def __init__(self, index: int):
        self.index, self.proc, self.lines = index, None, []

    def start(self):
        try:
            self.proc = subprocess.Popen(
                ["nvidia-smi", f"--id={self.index}", f"--query-gpu={self.Q}", "--format=csv,noheader,nounits", "-lms", "20"],
                stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
            self.thread = threading.Thread(target=self._read, daemon=True)
            self.thread.start()
        except OSError:
            self.proc = None

    def _read(self):
        for line in self.proc.stdout:
            self.lines.append((time.perf_counter(), line.strip()))

    def stop(self, t0=None, t1=None):
        if self.proc is None:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        self.proc.terminate()
        try:
            self.proc.wait(timeout=5)
        except subprocess.TimeoutExpired:
            self.proc.kill()
        sm, smax, reasons, power = [], [], set(), []
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        lines = [ln for t, ln in self.lines if t0 is None or (t0 <= t <= t1 + 0.02)]
        if not lines:  # region shorter than one sampling period: the samples nearest to it
            lines = [ln for _, ln in self.lines[-3:]]
        for ln in lines:
            f = [x.strip() for x in ln.split(",")]
            if len(f) < 7:
                continue
            try:
                sm.append(float(f[0]))
                smax.append(float(f[1]))
                power.append(float(f[2]))
            except ValueError:
                continue
            for nm, v in zip(names, f[3:7]):
                if v.lower().startswith("active"):
                    reasons.add(nm)
        return {"sm_mhz": float(np.median(sm)) if sm else None, "sm_max_mhz": max(smax) if smax else None,
                "power_w_max": max(power) if power else None, "samples": len(sm), "reasons": sorted(reasons)}


def oracle_sample(wl, n_sn_sample: int):
    """First n_sn_sample supernovae of the workload as their own Workload (bounded CPU sample)."""
    n = min(n_sn_sample, wl.n_sn)
    hi = int(wl.obs_offset[n])
    ns = wl.n_samples
    sub = workloads.Workload(
        config=wl.config, name=wl.name + f"[:{n}]", model=wl.model, bands=wl.bands, n_sn=n, n_samples=ns,
        obs_offset=wl.obs_offset[:n + 1].copy(), time=wl.time[:hi], band=wl.band[:hi], zp=wl.zp[:hi], z=wl.z[:n],
        theta_true={k: v[:n] for k, v in wl.theta_true.items()}, theta={k: v[:n * ns] for k, v in wl.theta.items()},
        noise=wl.noise[:hi])
    return sub


def oracle_sample_samples(wl, k: int):
    """Keep the first k parameter samples of every supernova (config 3 has one SN, 65536 samples)."""
    k = min(k, wl.n_samples)
    th = {key: v.reshape(wl.n_sn, wl.n_samples)[:, :k].ravel().copy() for key, v in wl.theta.items()}
    return workloads.Workload(
        config=wl.config, name=wl.name + f"[samples :{k}]", model=wl.model, bands=wl.bands, n_sn=wl.n_sn,
        n_samples=k, obs_offset=wl.obs_offset, time=wl.time, band=wl.band, zp=wl.zp, z=wl.z,
        theta_true=wl.theta_true, theta=th, noise=wl.noise)


def time_oracle(wl, evals_target: int, steps: int, warmup: int, threads=None):
    """Time the oracle, as it stands, on a bounded prefix of the workload (host cores of this box;
    `threads` = None: all of them)."""
    import oracle

    kw = {"threads": int(threads) if threads else len(os.sched_getaffinity(0))}

    if wl.n_samples > 1:
        k = max(1, min(wl.n_samples, evals_target // max(wl.n_obs_total, 1)))
        sub = oracle_sample_samples(wl, k)
        sample = f"first {k} of {wl.n_samples} parameter samples of {wl.name} ({sub.n_evals} evals)"
    else:
        n = max(1, min(wl.n_sn, evals_target // max(int(wl.meta.get('n_obs_per_sn', 1)), 1)))
        sub = oracle_sample(wl, n)
        sample = f"first {n} of {wl.n_sn} supernovae of {wl.name} ({sub.n_evals} evals)"
    # the oracle's own flux at theta_true provides the photometry of its sample
    true = oracle.run_workload(sub, theta={k_: v.copy() for k_, v in sub.theta_true.items()})["flux"]
    workloads.attach_data(sub, true)
    for _ in range(warmup):
        oracle.run_workload(sub, want_flux=True, want_chi2=True, **kw)
    t = []
    for _ in range(steps):
        t0 = time.perf_counter()
        oracle.run_workload(sub, want_flux=True, want_chi2=True, **kw)
        t.append(time.perf_counter() - t0)
    sec = float(np.mean(t))
    return sub.n_evals / sec, sec, oracle.num_threads(), sample


def fp32_peak_tflops(stream_ptr: int):
    import ctypes as C

    path = os.path.join(ROOT, "paper_2504_08081_b200", "libsbprobe.so")
    L = C.CDLL(path)
    L.sbp_fma_peak.restype = C.c_int
    L.sbp_fma_peak.argtypes = [C.c_int, C.c_int, C.c_void_p, C.POINTER(C.c_double), C.POINTER(C.c_double)]
    tf, ms = C.c_double(), C.c_double()
    rc = L.sbp_fma_peak(2000, 5, stream_ptr, C.byref(tf), C.byref(ms))
    if rc != 0:
        raise RuntimeError(f"sbp_fma_peak failed ({rc})")
    return tf.value, ms.value


def run_reference(args):
    """--impl reference: the fp64 CPU oracle (this tier's reference arm), rank 0 only."""
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return 0
    wl = workloads.make_workload(args.config)
    steps, warmup = max(args.steps, 1), max(args.warmup, 0)
    import oracle

    pilot_target = 4000
    v_pilot, _, cores, _ = time_oracle(wl, pilot_target, 1, 0)
    budget_s = 150.0 / (steps + warmup)
    evals_target = int(max(pilot_target, min(v_pilot * budget_s, wl.n_evals)))
    value, sec, cores, sample = time_oracle(wl, evals_target, steps, warmup)
    line = {
        "impl": "reference", "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": args.gpus, "steps": steps,
        "warmup": warmup, "ms_per_step": sec * 1e3, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
        "dtype": "f64", "data": "synthetic",
        "config": {"workload": wl.name, "n_sn": wl.n_sn, "n_samples": wl.n_samples, "n_evals": wl.n_evals,
                   "mode": "chi2", "note": "fp64 CPU oracle on a bounded sample per step"},
        "cpu_baseline": {"value": value, "unit": UNIT, "cores": cores, "kind": "oracle", "sample": sample},
        "e2e": {"value": value, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0,
    }
    print(json.dumps(line))
    return 0


def run_fit(args):
    """--mode fit: the batched device-resident L-BFGS fit (sb_fit_lbfgs; PAPER.md:17 fmin_bfgs.py) on
    BASELINE.json configs[3] (4096 supernovae x 100 observations, perturbed start).  A step = one whole fit of
    every supernova: --fit-evals batched chi^2 + gradient evaluations and lane updates, no host sync.
    e2e = sb_fit_lbfgs_host on pinned host buffers; the oracle optimiser (oracle/lbfgs.py) is timed beside it
    on a bounded sample."""
    import torch

    import paper_2504_08081_b200 as sb

    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    local_rank = int(os.environ.get("LOCAL_RANK", "0"))
    if not torch.cuda.is_available():
        raise RuntimeError("bench.py needs a CUDA device: there is no CPU fallback")
    torch.cuda.set_device(local_rank)
    dev = torch.device("cuda", local_rank)
    dist = None
    if world > 1:
        import torch.distributed as dist

        dist.init_process_group("nccl", device_id=dev)
    config = 4 if args.config == 5 else args.config
    steps, warmup = max(min(args.steps, 50), 1), max(min(args.warmup, 5), 3)
    wl = workloads.make_workload(config, seed_offset=rank)
    md, bd = wl.model, wl.bands
    model = sb.sb_load_model(md["phase"], md["wave"], md["m0"], md["m1"], md["cl_coef"], md["cl_wave_b"],
                             md["cl_wave_v"], md["cl_lo"], md["cl_hi"])
    bands = sb.sb_load_bandpasses(bd["offset"], bd["wave"], bd["trans"])
    ft = torch.float32
    n, n_tot = wl.n_sn, wl.n_obs_total

    def pin(a, dtype):
        return torch.as_tensor(np.ascontiguousarray(a)).to(dtype).pin_memory()

    h = {"obs_offset": pin(wl.obs_offset, torch.int32), "time": pin(wl.time, ft), "band": pin(wl.band, torch.int32),
         "zp": pin(wl.zp, ft), "z": pin(wl.z, ft)}
    for k in ("x0", "x1", "c", "t0"):
        h[k] = pin(wl.theta[k], ft)
    d = {k: v.to(dev) for k, v in h.items()}
    tt = {k: torch.as_tensor(wl.theta_true[k]).to(dev) for k in ("x0", "x1", "c", "t0")}
    true_flux = torch.empty(n_tot, dtype=ft, device=dev)
    sb.sb_bandflux(model, bands, dtype=sb.SB_F32, n_sn=n, n_samples=1, n_obs_total=n_tot, obs_offset=d["obs_offset"],
                   time=d["time"], band=d["band"], zp=d["zp"], z=d["z"], out_flux=true_flux, **tt)
    torch.cuda.synchronize()
    workloads.attach_data(wl, true_flux.double().cpu().numpy())
    h["flux"], h["fluxerr"] = pin(wl.flux, ft), pin(wl.fluxerr, ft)
    d["flux"], d["fluxerr"] = h["flux"].to(dev), h["fluxerr"].to(dev)
    pack = sb.sb_pack_observations(model, bands, dtype=sb.SB_F32, n_sn=n, z=d["z"])
    opts = dict(max_eval=args.fit_evals, ftol=1e-7)
    common = dict(dtype=sb.SB_F32, n_sn=n, n_samples=1, n_obs_total=n_tot)
    o = dict(out_theta=torch.empty((n, 4), dtype=ft, device=dev), out_chi2=torch.empty(n, dtype=ft, device=dev),
             out_status=torch.empty(n, dtype=torch.int32, device=dev), out_n_iter=torch.empty(n, dtype=torch.int32, device=dev),
             out_n_eval=torch.empty(n, dtype=torch.int32, device=dev))
    ho = {k: torch.empty_like(v, device="cpu").pin_memory() for k, v in o.items()}
    launches = [0]

    def step():
        sb.sb_fit_lbfgs(model, bands, **d, **o, pack=pack, **common, **opts)
        launches[0] = sb.last_launch_count()

    def barrier():
        if dist is not None:
            dist.barrier()
        torch.cuda.synchronize()

    sampler = ClockSampler(local_rank)
    sampler.start()
    for _ in range(warmup):
        step()
    barrier()
    ev = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)) for _ in range(steps)]
    wall0 = time.perf_counter()
    for a, b in ev:
        a.record()
        step()
        b.record()
    barrier()
    clocks = sampler.stop(wall0, time.perf_counter())
    total_ms = float(sum(a.elapsed_time(b) for a, b in ev))
    if dist is not None:
        tmax = torch.tensor([total_ms], dtype=torch.float64, device=dev)
        dist.all_reduce(tmax, op=dist.ReduceOp.MAX)
        total_ms = float(tmax.item())
    ms_per_step = total_ms / steps
    n_eval = o["out_n_eval"].cpu().numpy().astype(np.int64)
    status = o["out_status"].cpu().numpy()
    chi2 = o["out_chi2"].double().cpu().numpy()
    e2e_steps = min(steps, 10)
    for _ in range(2):
        sb.sb_fit_lbfgs_host(model, bands, **h, **ho, **common, **opts)
    barrier()
    t0 = time.perf_counter()
    for _ in range(e2e_steps):
        sb.sb_fit_lbfgs_host(model, bands, **h, **ho, **common, **opts)
    e2e_ms = (time.perf_counter() - t0) * 1e3 / e2e_steps
    if dist is not None:
        tmax = torch.tensor([e2e_ms], dtype=torch.float64, device=dev)
        dist.all_reduce(tmax, op=dist.ReduceOp.MAX)
        e2e_ms = float(tmax.item())
    if rank != 0:
        if dist is not None:
            dist.destroy_process_group()
        return 0
    cpu = None
    if world == 1 and not args.no_cpu_baseline:
        import oracle
        from oracle import lbfgs

        k = 24  # bounded sample: the first 24 supernovae, one lane at a time on one host core
        sub = oracle_sample(wl, k)
        true = oracle.run_workload(sub, theta={k_: v.copy() for k_, v in sub.theta_true.items()})["flux"]
        workloads.attach_data(sub, true)
        t0 = time.perf_counter()
        ref = lbfgs.fit_workload(sub, round_theta_to=np.float32, **opts)
        sec = time.perf_counter() - t0
        cpu = {"value": k / sec, "unit": "fits/s", "cores": 1, "kind": "oracle (oracle/lbfgs.py over the fp64 oracle)",
               "sample": f"first {k} of {wl.n_sn} supernovae of {wl.name}", "seconds": sec,
               "evaluations_per_sec": float(ref["n_eval"].sum()) / sec, "mean_n_eval": float(ref["n_eval"].mean())}
    in_bytes = sum(v.numel() * v.element_size() for v in h.values())
    out_bytes = sum(v.numel() * v.element_size() for v in ho.values())
    line = {
        "metric": "lbfgs_fits_per_sec", "value": n * world / (ms_per_step * 1e-3), "unit": "fits/s", "n_gpus": world,
        "steps": steps, "warmup": warmup, "ms_per_step": ms_per_step, "higher_is_better": True, "scaling": "weak",
        "vs_baseline": None, "dtype": "f32 evaluations, f64 optimiser state", "data": "synthetic",
        "config": {"workload": wl.name, "n_sn": n, "n_obs_total": n_tot, "mode": "fit", "max_eval": args.fit_evals,
                   "ftol": opts["ftol"], "memory": 8, "pack": True,
                   "evaluations_per_sec": float(n_eval.sum()) * world / (ms_per_step * 1e-3),
                   "bandflux_grad_evals_per_sec": float((n_eval * np.diff(wl.obs_offset)).sum()) * world / (ms_per_step * 1e-3),
                   "mean_n_eval": float(n_eval.mean()), "converged_frac": float(np.mean(status == 1)),
                   "median_chi2": float(np.median(chi2)), "parallelism": f"dp{world} (independent shards)"},
        "e2e": {"value": n * world / (e2e_ms * 1e-3), "unit": "fits/s", "h2d_bytes_per_step": in_bytes,
                "d2h_bytes_per_step": out_bytes, "ms_per_step": e2e_ms, "steps": e2e_steps, "call": "sb_fit_lbfgs_host"},
        "gpu_launches": launches[0] * steps, "clocks": clocks, "cpu_baseline": cpu,
    }
    print(json.dumps(line))
    if dist is not None:
        dist.destroy_process_group()
    return 0


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=200)
    ap.add_argument("--warmup", type=int, default=10)
    ap.add_argument("--config", type=int, default=5, choices=[1, 2, 3, 4, 5])
    ap.add_argument("--mode", default="chi2", choices=["chi2", "grad", "fit"],
                    help="chi2: sb_chi2 (default); grad: sb_bandflux_grad; fit: sb_fit_lbfgs (batched L-BFGS, config 4 shape)")
    ap.add_argument("--pack", action="store_true",
                    help="time the calls with an sb_pack_observations pack (built once, outside the timed region)")
    ap.add_argument("--band-jitter", type=float, default=0.0,
                    help="non-uniform band grids: interior grid points moved by U(-j, j) x step (workloads.jitter_band_grids)")
    ap.add_argument("--fit-evals", type=int, default=40, help="--mode fit: evaluations (steps) per lane")
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--form", default="auto", choices=["auto", "direct", "grouped", "tiled"],
                    help="formulation (include/saltband.h SB_FORM_*): auto = the library's choice")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--cpu-evals", type=int, default=2400000,
                    help="evals in the cpu_baseline sample (about 15 s of the fp64 oracle on 16 host threads)")
    args = ap.parse_args()
    if args.impl == "reference":
        return run_reference(args)
    if args.mode == "fit":
        return run_fit(args)

    import torch

    import paper_2504_08081_b200 as sb

    world = int(os.environ.get("WORLD_SIZE", "1"))
    rank = int(os.environ.get("RANK", "0"))
    local_rank = int(os.environ.get("LOCAL_RANK", "0"))
    if not torch.cuda.is_available():
        raise RuntimeError("bench.py needs a CUDA device: there is no CPU fallback")
    torch.cuda.set_device(local_rank)
    dev = torch.device("cuda", local_rank)
    dist = None
    if world > 1:
        import torch.distributed as dist

        dist.init_process_group("nccl", device_id=dev)
    steps, warmup = max(args.steps, 1), max(args.warmup, 3)
    grad = args.mode == "grad"

    # ---- workload shard of this rank (weak scaling: one full config per GPU)
    wl = workloads.make_workload(args.config, seed_offset=rank, band_jitter=args.band_jitter)
    md, bd = wl.model, wl.bands
    model = sb.sb_load_model(md["phase"], md["wave"], md["m0"], md["m1"], md["cl_coef"], md["cl_wave_b"],
                             md["cl_wave_v"], md["cl_lo"], md["cl_hi"])
    bands = sb.sb_load_bandpasses(bd["offset"], bd["wave"], bd["trans"])
    n_tot, ns, n_units, n_ev = wl.n_obs_total, wl.n_samples, wl.n_sn * wl.n_samples, wl.n_evals
    ft = torch.float32

    def pin(a, dtype):
        t = torch.as_tensor(np.ascontiguousarray(a)).to(dtype)
        return t.pin_memory()

    h = {"obs_offset": pin(wl.obs_offset, torch.int32), "time": pin(wl.time, ft), "band": pin(wl.band, torch.int32),
         "zp": pin(wl.zp, ft), "z": pin(wl.z, ft)}
    for k in ("x0", "x1", "c", "t0"):
        h[k] = pin(wl.theta[k], ft)
    d = {k: v.to(dev, non_blocking=True) for k, v in h.items()}
    form_bits = {"auto": 0, "direct": sb.SB_FORM_DIRECT, "grouped": sb.SB_FORM_GROUPED, "tiled": sb.SB_FORM_TILED}[args.form]
    common = dict(dtype=sb.SB_F32 | form_bits, n_sn=wl.n_sn, n_samples=ns, n_obs_total=n_tot)

    # photometry: the CUDA path's own flux at theta_true + seeded noise (inputs of the timed call only)
    tt = {k: torch.as_tensor(wl.theta_true[k]).to(dev) for k in ("x0", "x1", "c", "t0")}
    true_flux = torch.empty(n_tot, dtype=ft, device=dev)
    sb.sb_bandflux(model, bands, dtype=sb.SB_F32, n_sn=wl.n_sn, n_samples=1, n_obs_total=n_tot,
                   obs_offset=d["obs_offset"], time=d["time"], band=d["band"], zp=d["zp"], z=d["z"], out_flux=true_flux, **tt)
    torch.cuda.synchronize()
    workloads.attach_data(wl, true_flux.double().cpu().numpy())
    h["flux"], h["fluxerr"] = pin(wl.flux, ft), pin(wl.fluxerr, ft)
    d["flux"], d["fluxerr"] = h["flux"].to(dev), h["fluxerr"].to(dev)

    # optional pack (include/saltband.h: sb_pack_observations): z order and item geometry, built once
    pack = sb.sb_pack_observations(model, bands, dtype=sb.SB_F32, n_sn=wl.n_sn, z=d["z"])
    torch.cuda.synchronize()
    use_pack = [bool(args.pack)]

    o_flux = torch.empty(n_ev, dtype=ft, device=dev)
    o_chi = torch.empty(n_units, dtype=ft, device=dev)
    o_dflux = torch.empty(n_ev * 4, dtype=ft, device=dev) if grad else None
    o_dchi = torch.empty(n_units * 4, dtype=ft, device=dev) if grad else None
    launches_per_step = [0]
    form_ran = [""]

    def step(t):
        pk = pack if use_pack[0] else None
        if grad:
            sb.sb_bandflux_grad(model, bands, obs_offset=t["obs_offset"], time=t["time"], band=t["band"], zp=t["zp"],
                                z=t["z"], x0=t["x0"], x1=t["x1"], c=t["c"], t0=t["t0"], flux=t["flux"],
                                fluxerr=t["fluxerr"], out_flux=o_flux, out_dflux=o_dflux, out_chi2=o_chi,
                                out_dchi2=o_dchi, pack=pk, **common)
        else:
            sb.sb_chi2(model, bands, obs_offset=t["obs_offset"], time=t["time"], band=t["band"], zp=t["zp"], z=t["z"],
                       x0=t["x0"], x1=t["x1"], c=t["c"], t0=t["t0"], flux=t["flux"], fluxerr=t["fluxerr"],
                       out_chi2=o_chi, out_flux=o_flux, pack=pk, **common)
        launches_per_step[0] = sb.last_launch_count()
        form_ran[0] = sb.last_form()

    in_bytes = sum(v.numel() * v.element_size() for v in h.values())
    out_bytes = o_flux.numel() * 4 + o_chi.numel() * 4 + (o_dflux.numel() * 4 + o_dchi.numel() * 4 if grad else 0)
    l2_bytes = 126 * 1024 * 1024
    need_flush = (in_bytes + out_bytes) <= l2_bytes
    flush_buf = torch.empty(256 * 1024 * 1024, dtype=torch.uint8, device=dev) if need_flush else None

    def barrier():
        if dist is not None:
            dist.barrier()
        torch.cuda.synchronize()

    # ---- device-resident timing: K steps, CUDA events per step on the launching (current) stream
    sampler = ClockSampler(local_rank)
    sampler.start()
    for _ in range(warmup):
        step(d)
    barrier()
    ev = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)) for _ in range(steps)]
    wall0 = time.perf_counter()
    for a, b in ev:
        if need_flush:
            flush_buf.fill_(1)
        a.record()
        step(d)
        b.record()
    barrier()
    wall1 = time.perf_counter()
    wall = wall1 - wall0
    clocks = sampler.stop(wall0, wall1)
    per_step_ms = np.array([a.elapsed_time(b) for a, b in ev])
    total_ms = float(per_step_ms.sum())
    if dist is not None:
        tmax = torch.tensor([total_ms], dtype=torch.float64, device=dev)
        dist.all_reduce(tmax, op=dist.ReduceOp.MAX)
        total_ms = float(tmax.item())
    ms_per_step = total_ms / steps
    value = n_ev * world * steps / (total_ms * 1e-3)
    launches_timed = launches_per_step[0]

    # ---- the same call with a pack (or without, if --pack): observations and redshifts are static over the
    # thousands of calls of a fit or a sampling run, so the theta-independent work can be
    # done once; reported beside the headline value, which times everything a bare call launches
    use_pack[0] = not use_pack[0]
    alt_steps = min(steps, 50)
    for _ in range(3):
        step(d)
    barrier()
    ev2 = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)) for _ in range(alt_steps)]
    for a, b in ev2:
        if need_flush:
            flush_buf.fill_(1)
        a.record()
        step(d)
        b.record()
    barrier()
    alt_ms = float(np.mean([a.elapsed_time(b) for a, b in ev2]))
    alt = {"pack": use_pack[0], "ms_per_step": alt_ms, "value": n_ev / (alt_ms * 1e-3), "steps": alt_steps,
           "gpu_launches_per_step": launches_per_step[0], "note": "this rank only"}
    use_pack[0] = not use_pack[0]

    # ---- end to end: the host-buffer C-ABI call (sb_chi2_host / sb_bandflux_grad_host) on pinned host
    # inputs and outputs: every step copies all inputs host -> device and all results device -> host
    # (chunked, overlapped with the kernels, on the library's own streams) and returns when complete
    h_flux_out = torch.empty(n_ev, dtype=ft).pin_memory()
    h_chi_out = torch.empty(n_units, dtype=ft).pin_memory()
    h_dflux_out = torch.empty(n_ev * 4, dtype=ft).pin_memory() if grad else None
    h_dchi_out = torch.empty(n_units * 4, dtype=ft).pin_memory() if grad else None

    def e2e_step():
        if grad:
            sb.sb_bandflux_grad_host(model, bands, obs_offset=h["obs_offset"], time=h["time"], band=h["band"],
                                     zp=h["zp"], z=h["z"], x0=h["x0"], x1=h["x1"], c=h["c"], t0=h["t0"],
                                     flux=h["flux"], fluxerr=h["fluxerr"], out_flux=h_flux_out, out_dflux=h_dflux_out,
                                     out_chi2=h_chi_out, out_dchi2=h_dchi_out, **common)
        else:
            sb.sb_chi2_host(model, bands, obs_offset=h["obs_offset"], time=h["time"], band=h["band"], zp=h["zp"],
                            z=h["z"], x0=h["x0"], x1=h["x1"], c=h["c"], t0=h["t0"], flux=h["flux"],
                            fluxerr=h["fluxerr"], out_chi2=h_chi_out, out_flux=h_flux_out, **common)

    e2e_steps = min(steps, 20)
    for _ in range(2):
        e2e_step()
    barrier()
    t_e2e = time.perf_counter()  # the call is synchronous: host clock around K calls, device idle before and after
    for _ in range(e2e_steps):
        e2e_step()
    torch.cuda.synchronize()
    e2e_ms = (time.perf_counter() - t_e2e) * 1e3
    if dist is not None:
        tmax = torch.tensor([e2e_ms], dtype=torch.float64, device=dev)
        dist.all_reduce(tmax, op=dist.ReduceOp.MAX)
        e2e_ms = float(tmax.item())
    e2e_value = n_ev * world * e2e_steps / (e2e_ms * 1e-3)
    d2h = (h_flux_out.numel() + h_chi_out.numel() + (h_dflux_out.numel() + h_dchi_out.numel() if grad else 0)) * 4

    if rank != 0:
        if dist is not None:
            dist.destroy_process_group()
        return 0

    # ---- roofline of the (single) kernel: ALU-bound, against the FP32 FMA peak measured here
    # which formulation ran: the grouped kernel launches a one-CTA z-order kernel before the main one
    form_run = form_ran[0]
    flops_ours, flops_survey, mean_in, mean_cell = flops_per_call(wl, grad, form_run)
    # events bracket the step's launches: the main kernel plus, in the grouped form, the one-CTA
    # z-order kernel (< 1 % of the step, profiles/)
    kernel_ms = float(np.mean(per_step_ms))
    try:
        peak_tf, _ = fp32_peak_tflops(torch.cuda.current_stream().cuda_stream)
        peak_src = "measured: FFMA-chain microbenchmark (csrc/sb_probe.cu) in this run"
    except Exception as exc:  # pragma: no cover
        peak_tf, peak_src = 148 * 128 * 2 * 1.965e9 * 1e-12, f"nominal 148 SM x 128 lanes x 2 x 1.965 GHz ({exc})"
    model_tf = flops_ours / (kernel_ms * 1e-3) * 1e-12
    algo_bytes = in_bytes + out_bytes
    # fraction = min(A, B) / peak, A = executed-model flops (above), B = FP32 flops
    # counted by ncu for one launch of this kernel on this workload (SASS opcode table of the committed
    # `ncu --set full` capture, profiles/traffic.json; packed FFMA2/FMUL2/FADD2 count twice) over the time
    # measured here.  B guards against an inflated model, A against counting padded or repeated work.
    cap = _ncu_capture(form_run, grad, wl.name)
    counted = cap.get("counted_fp32_flop")
    counted_tf = counted / (kernel_ms * 1e-3) * 1e-12 if counted else None
    achieved = min(model_tf, counted_tf) if counted_tf else model_tf
    roofline = {
        "bound": "alu", "achieved": achieved, "peak": peak_tf, "unit": "TFLOP/s", "frac": achieved / peak_tf,
        "model": model_tf, "counted": counted_tf, "counted_flop_per_launch": counted,
        "counted_source": cap.get("source"),
        "traffic": cap.get("dram_bytes"),
        "kernel": {"grouped": "sb_hoist_kernel<fwd>", "tiled": "sb_nw_kernel<%s>" % ("grad" if grad else "fwd")}.get(
            form_run, "sb_fused_kernel<float,%s>" % ("grad" if grad else "fwd")),
        "form": form_run,
        "kernel_ms": kernel_ms, "flops_per_eval": flops_ours / n_ev, "peak_source": peak_src,
        "flop_model": {"grouped": "executed formulation (DESIGN.md): node-weight re-association, G_geom = G_col = "
                                  "observations per (unit, band) chunk (<= 8)",
                       "tiled": "executed formulation (DESIGN.md): node-weight re-association, G_geom = G_col = "
                                "observations per (unit, band)"}.get(
            form_run, "executed formulation (DESIGN.md): G_geom = G_col = 1"),
        "survey_direct_model": {"flops_per_eval": flops_survey / n_ev,
                                "evals_per_sec_at_half_peak": 0.5 * peak_tf * 1e12 / (flops_survey / n_ev),
                                "note": "SURVEY.md 8(d) G = 1 model: a rate target for context (BASELINE.md section 3), "
                                        "not work this kernel executes"},
        "mean_in_range_samples": mean_in, "mean_cells": mean_cell,
        "hbm": {"algorithmic_bytes": algo_bytes, "achieved_gbs": algo_bytes / (kernel_ms * 1e-3) * 1e-9,
                "peak_gbs": _measured_peaks().get("hbm_gbs"),
                "note": "path is ALU-bound: HBM moves only the per-observation records"},
    }
    cpu = None
    if world == 1 and not args.no_cpu_baseline:
        v, sec, cores, sample = time_oracle(wl, args.cpu_evals, 1, 0)
        cpu = {"value": v, "unit": UNIT, "cores": cores, "kind": "oracle", "sample": sample, "seconds": sec}
        v1, sec1, _, sample1 = time_oracle(wl, max(args.cpu_evals // 48, 4000), 1, 0, threads=1)
        cpu["single_thread"] = {"value": v1, "unit": UNIT, "cores": 1, "sample": sample1, "seconds": sec1}
    line = {
        "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": steps, "warmup": warmup,
        "ms_per_step": ms_per_step, "ms_per_step_median": float(np.median(per_step_ms)),
        "ms_per_step_min": float(per_step_ms.min()), "higher_is_better": True, "scaling": "weak",
        "vs_baseline": None, "dtype": "f32", "data": "synthetic",
        "config": {"workload": wl.name, "n_sn": wl.n_sn, "n_samples": ns, "n_obs_total": n_tot, "n_evals": n_ev,
                   "mode": args.mode, "form": form_run, "pack": bool(args.pack), "band_jitter": args.band_jitter, "chi2_evals_per_sec": n_units * world * steps / (total_ms * 1e-3),
                   "l2": "inputs+outputs %.0f MB > 126 MB L2, no flush" % ((in_bytes + out_bytes) / 1e6) if not need_flush
                   else "L2 flushed (256 MB write) between timed steps", "parallelism": f"dp{world} (independent shards)"},
        "e2e": {"value": e2e_value, "unit": UNIT, "h2d_bytes_per_step": in_bytes, "d2h_bytes_per_step": d2h,
                "ms_per_step": e2e_ms / e2e_steps, "steps": e2e_steps,
                "call": "sb_bandflux_grad_host" if grad else "sb_chi2_host"},
        "gpu_launches": launches_timed * steps, "clocks": clocks, "roofline": roofline, "cpu_baseline": cpu,
        "with_pack" if not args.pack else "without_pack": alt, "wall_s_timed_region": wall,
    }
    print(json.dumps(line))
    if dist is not None:
        dist.destroy_process_group()
    return 0


def _ncu_capture(form: str, grad: bool, workload: str) -> dict:
    """Per-launch figures of the step's main kernel copied from the `ncu --set full` capture summarised
    under profiles/ (profiles/traffic.json): dram_bytes = dram__bytes_read.sum + dram__bytes_write.sum,
    counted_fp32_flop = FP32 flops from the SASS opcode table.  {} if this (formulation, mode, workload)
    has not been captured."""
    try:
        with open(os.path.join(ROOT, "profiles", "traffic.json")) as fh:
            tab = json.load(fh)
    except (OSError, ValueError):
        return {}
    ent = tab.get(f"{form}:{'grad' if grad else 'fwd'}:{workload}")
    return ent if isinstance(ent, dict) else {}


def _measured_peaks():
    try:
        with open(os.path.join(ROOT, "MEASURED_PEAKS.json")) as fh:
            return json.load(fh)
    except OSError:
        return {}


if __name__ == "__main__":
    sys.exit(main())
