"""-m gpu: the device-resident batched L-BFGS fit (include/saltband.h: sb_fit_lbfgs; PAPER.md:17
"fmin_bfgs.py ... optimisation via L-BFGS-B"; reading G16) against oracle/lbfgs.py, one lane at a
time on the CPU over the fp64 oracle's chi^2 and gradient.

* fp64 batches: the lane state machine is the oracle's, so the chi^2 trajectory must agree to rounding
  (1e-9 relative over the first accepted steps) and the final theta to 1e-6 of its scale;
* fp32 batches (production): the trajectory differs by the kernels' rounding, the minimum reached must
  not: final chi^2 within 1e-4 relative of the oracle's;
* noise-free photometry: theta_true is recovered; a box is honoured; a pack, the host-buffer call and a
  CUDA-graph replay change nothing; a stopped lane is never evaluated again."""
import numpy as np
import pytest

import oracle
import sbgpu
import workloads
from oracle import lbfgs

pytestmark = pytest.mark.gpu

KEYS = ("x0", "x1", "c", "t0")


def _prepare(n_sn, noise=True, config=4, **kw):
    wl = workloads.make_workload(config, n_sn=n_sn, **kw)
    true = oracle.run_workload(wl, theta={k: v.copy() for k, v in wl.theta_true.items()})["flux"]
    if not noise:
        wl.noise = np.zeros(wl.n_obs_total)
    workloads.attach_data(wl, true)
    return wl


def _gpu_fit(wl, *, fp64, trace_len=0, use_pack=False, host=False, handles=None, tiled=False, **opts):
    import torch

    import paper_2504_08081_b200 as sb

    ft = torch.float64 if fp64 else torch.float32
    dev = torch.device("cpu" if host else "cuda:0")
    model, bands = handles if handles is not None else sbgpu.load_handles(wl)
    f = lambda a: torch.as_tensor(np.asarray(a, dtype=np.float64), dtype=ft).to(dev).contiguous()  # noqa: E731
    i = lambda a: torch.as_tensor(np.asarray(a, dtype=np.int32)).to(dev)  # noqa: E731
    n = wl.n_sn * wl.n_samples
    dtype = (sb.SB_F64 if fp64 else sb.SB_F32) | (sb.SB_FORM_TILED if tiled else 0)  # tiled: also for tiny batches
    args = dict(dtype=dtype, n_sn=wl.n_sn, n_samples=wl.n_samples, n_obs_total=wl.n_obs_total,
                obs_offset=i(wl.obs_offset), time=f(wl.time), band=i(wl.band), zp=f(wl.zp), z=f(wl.z),
                x0=f(wl.theta["x0"]), x1=f(wl.theta["x1"]), c=f(wl.theta["c"]), t0=f(wl.theta["t0"]),
                flux=f(wl.flux), fluxerr=f(wl.fluxerr))
    out = dict(out_theta=torch.full((n, 4), float("nan"), dtype=ft, device=dev),
               out_chi2=torch.full((n,), float("nan"), dtype=ft, device=dev),
               out_status=torch.full((n,), -1, dtype=torch.int32, device=dev),
               out_n_iter=torch.full((n,), -1, dtype=torch.int32, device=dev),
               out_n_eval=torch.full((n,), -1, dtype=torch.int32, device=dev))
    if trace_len:
        out["out_trace"] = torch.zeros((trace_len, n), dtype=torch.float64, device=dev)
    if host:
        sb.sb_fit_lbfgs_host(model, bands, **args, **out, **opts)
    else:
        if use_pack:
            args["pack"] = sb.sb_pack_observations(model, bands, dtype=sb.SB_F32, n_sn=wl.n_sn, z=args["z"])
        sb.sb_fit_lbfgs(model, bands, **args, **out, **opts)
        torch.cuda.synchronize()
    res = {k[4:]: v.cpu().numpy().astype(np.float64 if v.dtype.is_floating_point else np.int64) for k, v in out.items()}
    res["launches"], res["form"] = sb.last_launch_count(), sb.last_form()
    return res


def _scale(wl):
    return np.stack([np.abs(wl.theta["x0"].astype(np.float64)), np.ones(wl.n_sn), np.ones(wl.n_sn), np.ones(wl.n_sn)], axis=1)


def test_fp64_fit_follows_the_oracle_lane_by_lane(cuda_device):
    wl = _prepare(10)
    opts = dict(memory=8, max_eval=40, max_iter=1000, ftol=1e-10, gtol=0.0)
    ref = lbfgs.fit_workload(wl, **opts)
    got = _gpu_fit(wl, fp64=True, trace_len=41, **opts)
    assert got["form"] == "direct" and np.all(got["status"] != 0)
    for s in range(wl.n_sn):
        tr = ref["trace"][s]
        k = min(6, len(tr))  # start point and the first five accepted steps
        assert np.allclose(got["trace"][:k, s], tr[:k], rtol=1e-9, atol=0), (s, got["trace"][:k, s], tr[:k])
        assert np.all(np.diff(got["trace"][:got["n_iter"][s] + 1, s]) <= 0.0)  # Armijo: monotone chi^2
    assert np.all(np.abs(got["theta"] - ref["theta"]) <= 1e-6 * _scale(wl)), np.max(np.abs(got["theta"] - ref["theta"]) / _scale(wl), axis=0)
    assert np.allclose(got["chi2"], ref["chi2"], rtol=1e-9)
    # same decisions in every lane unless a comparison sat within rounding of its threshold
    assert np.mean(got["n_eval"] == ref["n_eval"]) >= 0.8 and np.mean(got["status"] == ref["status"]) >= 0.8


def test_fp32_fit_reaches_the_oracle_minimum(cuda_device):
    wl = _prepare(24)
    opts = dict(memory=8, max_eval=60, max_iter=1000, ftol=1e-7, gtol=0.0)
    ref = lbfgs.fit_workload(wl, round_theta_to=np.float32, **opts)
    for use_pack in (False, True):
        got = _gpu_fit(wl, fp64=False, use_pack=use_pack, trace_len=8, tiled=True, **opts)
        assert got["form"] == "tiled" and np.all(got["status"] != 0)
        assert np.allclose(got["chi2"], ref["chi2"], rtol=1e-4), np.max(np.abs(got["chi2"] / ref["chi2"] - 1))
        start = oracle.run_workload(wl, want_flux=False, want_chi2=True)["chi2"]
        assert np.allclose(got["trace"][0], start, rtol=1e-4)  # row 0 = chi^2 at the start point
        if use_pack:
            assert np.array_equal(got["theta"], first["theta"]) and np.array_equal(got["n_eval"], first["n_eval"])
        first = got
    # the fitted parameters agree where chi^2 constrains them: compare through the flux they predict
    th = {k: got["theta"][:, j] for j, k in enumerate(KEYS)}
    m_gpu = oracle.run_workload(wl, theta=th)["flux"]
    m_ref = oracle.run_workload(wl, theta={k: ref["theta"][:, j] for j, k in enumerate(KEYS)})["flux"]
    sig = wl.fluxerr.astype(np.float64)
    assert np.max(np.abs(m_gpu - m_ref) / sig) < 0.05  # a twentieth of the measurement error


def test_noise_free_fit_recovers_theta_true(cuda_device):
    wl = _prepare(64, noise=False)
    got = _gpu_fit(wl, fp64=False, use_pack=True, max_eval=80, ftol=0.0)
    tt = np.stack([wl.theta_true[k].astype(np.float64) for k in KEYS], axis=1)
    scale = np.stack([np.abs(tt[:, 0]), np.ones(wl.n_sn), np.ones(wl.n_sn), np.ones(wl.n_sn)], axis=1)
    start = oracle.run_workload(wl, want_flux=False, want_chi2=True)["chi2"]
    assert np.all(got["chi2"] <= 1e-5 * start)  # fp32 model fluxes: chi^2 floor ~ n_obs (1e-5 / 0.05)^2
    assert np.all(np.abs(got["theta"] - tt) <= 2e-3 * scale), np.max(np.abs(got["theta"] - tt) / scale, axis=0)


def test_box_is_honoured_and_matches_the_oracle(cuda_device):
    wl = _prepare(8)
    lo, hi = np.array([0.0, -0.2, -0.02, -1.0]), np.array([1.0, 0.2, 0.02, 1.0])
    got = _gpu_fit(wl, fp64=True, max_eval=40, ftol=1e-10, lo=lo, hi=hi)
    assert np.all(got["theta"] >= lo - 1e-15) and np.all(got["theta"] <= hi + 1e-15)
    model, bands = oracle.Model.from_dict(wl.model), oracle.Bands.from_dict(wl.bands)
    for s in range(wl.n_sn):  # the same lane in the oracle, bounds in its scaled variables
        sub = workloads.subset(wl, [s])
        sc = np.array([float(wl.theta["x0"][s]), 1.0, 1.0, 1.0])
        ref = lbfgs.fit_workload(sub, max_eval=40, ftol=1e-10, lo=lo / sc, hi=hi / sc)
        assert np.allclose(got["theta"][s], ref["theta"][0], rtol=1e-6, atol=1e-9 * sc), (s, got["theta"][s], ref["theta"][0])
    assert np.any(got["theta"][:, 1:] == lo[1:]) or np.any(got["theta"][:, 1:] == hi[1:])  # some bound is active


def test_host_call_graph_replay_and_budget(cuda_device):
    import torch

    import paper_2504_08081_b200 as sb

    wl = _prepare(300)
    handles = sbgpu.load_handles(wl)
    opts = dict(max_eval=25, ftol=1e-6)
    dev = _gpu_fit(wl, fp64=False, use_pack=True, handles=handles, **opts)
    host = _gpu_fit(wl, fp64=False, host=True, handles=handles, **opts)
    for k in ("theta", "chi2", "status", "n_iter", "n_eval"):
        assert np.array_equal(dev[k], host[k]), k
    assert np.all(dev["n_eval"] <= 25) and np.all((dev["status"] >= 1) & (dev["status"] <= 3))
    assert np.all(dev["n_eval"][dev["status"] == 3] == 25)  # exhausted lanes used the whole budget
    # steps: 1 init + per step (evaluation kernel + update kernel) [+ pack build in the host call]
    assert dev["launches"] == 1 + 2 * 25
    # the whole fit is stream-ordered (no synchronisation, no allocation once warm): capture and replay
    ft = torch.float32
    f = lambda a: torch.as_tensor(np.asarray(a, dtype=np.float32)).to(cuda_device)  # noqa: E731
    i = lambda a: torch.as_tensor(np.asarray(a, dtype=np.int32)).to(cuda_device)  # noqa: E731
    args = dict(dtype=sb.SB_F32, n_sn=wl.n_sn, n_samples=1, n_obs_total=wl.n_obs_total, obs_offset=i(wl.obs_offset),
                time=f(wl.time), band=i(wl.band), zp=f(wl.zp), z=f(wl.z), x0=f(wl.theta["x0"]), x1=f(wl.theta["x1"]),
                c=f(wl.theta["c"]), t0=f(wl.theta["t0"]), flux=f(wl.flux), fluxerr=f(wl.fluxerr))
    args["pack"] = sb.sb_pack_observations(handles[0], handles[1], dtype=sb.SB_F32, n_sn=wl.n_sn, z=args["z"])
    theta = torch.zeros((wl.n_sn, 4), dtype=ft, device=cuda_device)
    chi2 = torch.zeros(wl.n_sn, dtype=ft, device=cuda_device)
    stream = torch.cuda.Stream()
    with torch.cuda.stream(stream):
        sb.sb_fit_lbfgs(*handles, **args, out_theta=theta, out_chi2=chi2, **opts)  # warm: workspace allocated
        stream.synchronize()
        graph = torch.cuda.CUDAGraph()
        theta.zero_()
        with torch.cuda.graph(graph, stream=stream):
            sb.sb_fit_lbfgs(*handles, **args, out_theta=theta, out_chi2=chi2, **opts)
        theta.zero_()
        graph.replay()
    stream.synchronize()
    assert np.array_equal(theta.cpu().numpy().astype(np.float64), dev["theta"])
    assert np.array_equal(chi2.cpu().numpy().astype(np.float64), dev["chi2"])


def test_fp32_fit_with_the_default_options_converges(cuda_device):
    """sb_fit_default_opts (ftol 1e-12, gtol 0, 60 evaluations) in an SB_F32 batch: chi^2 comes back in fp32, so
    the library raises that ftol to 2^-21 (include/saltband.h).  Without the floor a lane near its minimum
    burns its budget on halvings and ends stalled or exhausted; with it the lanes stop CONVERGED at the minimum
    the oracle finds."""
    wl = _prepare(48)
    got = _gpu_fit(wl, fp64=False, use_pack=True)  # every option left at the library's default
    assert np.all(got["status"] != 0)
    assert np.mean(got["status"] == 1) >= 0.9, np.bincount(got["status"].astype(int), minlength=4)
    ref = lbfgs.fit_workload(wl, round_theta_to=np.float32, memory=8, max_eval=60, max_iter=1000, ftol=2.0 ** -21, gtol=0.0)
    assert np.allclose(got["chi2"], ref["chi2"], rtol=1e-4), np.max(np.abs(got["chi2"] / ref["chi2"] - 1))
    # an explicit zero still switches the test off: no lane converges by ftol, every lane spends its budget or stalls
    off = _gpu_fit(wl, fp64=False, use_pack=True, ftol=0.0, max_eval=30)
    assert not np.any(off["status"] == 1)


def test_fp32_box_holds_exactly_after_rounding(cuda_device):
    """Bounds that are not fp32 numbers (-0.3, 0.1, 1e-5 x0 scale): every returned theta must satisfy
    lo <= theta <= hi exactly as fp32 values compared in fp64, although the lane projects in scaled fp64
    variables and the result is rounded to fp32 afterwards."""
    wl = _prepare(64)
    x0 = wl.theta["x0"].astype(np.float64)
    lo = np.array([0.3 * x0.min(), -0.3, -0.03, -0.7])
    hi = np.array([1.7 * x0.max(), 0.1, 0.03, 0.3])
    got = _gpu_fit(wl, fp64=False, use_pack=True, max_eval=40, ftol=1e-6, lo=lo, hi=hi)
    assert np.all(got["theta"] >= lo[None, :]) and np.all(got["theta"] <= hi[None, :])
    lo32, hi32 = np.float32(lo), np.float32(hi)
    edge = np.stack([lo32, hi32, np.nextafter(lo32, np.float32(np.inf)), np.nextafter(hi32, np.float32(-np.inf))]).astype(np.float64)
    at_bound = np.any(got["theta"][:, None, :] == edge[None, :, :], axis=1)
    assert at_bound[:, 1:].any()  # some bound is active, so the clamp was exercised
