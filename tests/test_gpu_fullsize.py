"""-m gpu parity at BASELINE.json's FULL sizes, in the launch configuration bench.py times (one
`sb_chi2` / `sb_bandflux_grad` call over the whole config, library's choice of formulation), on
SAMPLED units the oracle computes one by one (the oracle needs ~6 us per band sample, so the whole
of configs 3-5 would take minutes).  Photometry of the sampled units comes from the oracle's flux at
theta_true; the other units get seeded noise with unit errors (inputs only, never compared)."""
import numpy as np
import pytest

import oracle
import sbgpu
import workloads

pytestmark = pytest.mark.gpu


def _attach_sampled(wl, idx):
    """Photometry: oracle-derived on the sampled supernovae, seeded noise (sigma = 1) elsewhere."""
    sub = workloads.subset(wl, idx)
    true = oracle.run_workload(sub, theta={k: v.copy() for k, v in sub.theta_true.items()}, want_flux=True)["flux"]
    workloads.attach_data(sub, true)
    wl.flux = wl.noise.astype(np.float32)
    wl.fluxerr = np.ones(wl.n_obs_total, dtype=np.float32)
    for k, s in enumerate(idx):
        a, b = int(wl.obs_offset[s]), int(wl.obs_offset[s + 1])
        c, d = int(sub.obs_offset[k]), int(sub.obs_offset[k + 1])
        wl.flux[a:b], wl.fluxerr[a:b] = sub.flux[c:d], sub.fluxerr[c:d]
    return sub


def _gather_units(wl, idx, arr, per_obs):
    """Rows of a per-evaluation (per_obs) or per-unit output of the full call that belong to idx."""
    ns = wl.n_samples
    out = []
    for s in idx:
        if per_obs:
            out.append(arr[int(wl.obs_offset[s]) * ns:int(wl.obs_offset[s + 1]) * ns])
        else:
            out.append(arr[s * ns:(s + 1) * ns])
    return np.concatenate(out)


def _sample_indices(n, k, seed):
    rng = np.random.default_rng(seed)
    idx = np.unique(np.concatenate([[0, 1, n - 2, n - 1], rng.choice(n, size=min(k, n), replace=False)]))
    return idx[(idx >= 0) & (idx < n)]


@pytest.mark.parametrize("config,k", [(5, 2000), (4, 400), (2, 1024)])
def test_full_size_forward_sampled_units(cuda_device, config, k):
    wl = workloads.make_workload(config)  # full BASELINE.json size
    idx = _sample_indices(wl.n_sn, k, 77 + config)
    sub = _attach_sampled(wl, idx)
    ref = oracle.run_workload(sub, want_flux=True, want_chi2=True)
    got = sbgpu.run_gpu(wl, mode="chi2")
    assert got["launches"] >= 1 and got["form"] in ("tiled", "grouped", "direct")
    g_flux = _gather_units(wl, idx, got["flux"], True)
    g_chi = _gather_units(wl, idx, got["chi2"], False)
    tol = sbgpu.flux_tolerance(sub, ref["flux"], 1, False)
    err = np.abs(g_flux - ref["flux"])
    assert np.all(err <= tol), f"worst flux err/tol {np.max(err / np.maximum(tol, 1e-300)):.3g}"
    tolc = sbgpu.chi2_tolerance(sub, ref["flux"], tol, 1, False)
    assert np.all(np.abs(g_chi - ref["chi2"]) <= tolc)
    # properties that hold at any size: every output written, finite, chi^2 >= 0
    assert np.all(np.isfinite(got["flux"])) and np.all(np.isfinite(got["chi2"])) and np.all(got["chi2"] >= 0)
    # ALL units (also the groups without a sampled unit): the node-weight kernel against the direct
    # kernel, two exact re-associations of the same sums, each within the flux tolerance of the oracle
    assert got["form"] == "tiled"
    direct = sbgpu.run_gpu(wl, mode="chi2", form="direct")
    peak = sbgpu.unit_peaks(wl, direct["flux"], 1)
    tol_all = 2.0 * (1e-5 * np.abs(direct["flux"]) + 1e-9 * peak)
    err_all = np.abs(got["flux"] - direct["flux"])
    assert np.all(err_all <= tol_all), f"tiled vs direct worst ratio {np.max(err_all / np.maximum(tol_all, 1e-300)):.3g}"
    # with a pack (sb_pack_observations) the call gives bit-identical results
    packed = sbgpu.run_gpu(wl, mode="chi2", use_pack=True)
    assert np.array_equal(packed["flux"], got["flux"]) and np.array_equal(packed["chi2"], got["chi2"])


def test_full_size_config3_sampled_parameter_samples(cuda_device):
    wl = workloads.make_workload(3)  # 1 SN x 65536 samples x 50 obs
    ref_true = oracle.run_workload(wl, theta={k: v.copy() for k, v in wl.theta_true.items()}, want_flux=True)["flux"]
    workloads.attach_data(wl, ref_true)
    got = sbgpu.run_gpu(wl, mode="chi2")
    ks = np.unique(np.concatenate([[0, 1, wl.n_samples - 1], np.random.default_rng(5).choice(wl.n_samples, 400, replace=False)]))
    th = {k: v[ks].copy() for k, v in wl.theta.items()}
    ref = oracle.run_workload(wl, theta=th, want_flux=True, want_chi2=True)
    n_obs = wl.n_obs_total
    g_flux = got["flux"].reshape(wl.n_samples, n_obs)[ks].ravel()
    sub_like = workloads.Workload(config=3, name="c3 samples", model=wl.model, bands=wl.bands, n_sn=1, n_samples=len(ks),
                                  obs_offset=wl.obs_offset, time=wl.time, band=wl.band, zp=wl.zp, z=wl.z,
                                  theta_true=wl.theta_true, theta=th, noise=wl.noise, flux=wl.flux, fluxerr=wl.fluxerr)
    tol = sbgpu.flux_tolerance(sub_like, ref["flux"], len(ks), False)
    err = np.abs(g_flux - ref["flux"])
    assert np.all(err <= tol), f"worst flux err/tol {np.max(err / np.maximum(tol, 1e-300)):.3g}"
    tolc = sbgpu.chi2_tolerance(sub_like, ref["flux"], tol, len(ks), False)
    assert np.all(np.abs(got["chi2"][ks] - ref["chi2"]) <= tolc)
    assert np.all(np.isfinite(got["chi2"])) and np.all(got["chi2"] >= 0)


def test_full_size_config4_gradient_sampled_units(cuda_device):
    wl = workloads.make_workload(4)  # 4096 SN x 100 obs
    idx = _sample_indices(wl.n_sn, 96, 404)
    sub = _attach_sampled(wl, idx)
    ref = oracle.run_workload(sub, want_flux=True, want_chi2=True, want_dflux=True, want_dchi2=True)
    got = sbgpu.run_gpu(wl, mode="grad")
    g_flux = _gather_units(wl, idx, got["flux"], True)
    g_dflux = _gather_units(wl, idx, got["dflux"], True)
    g_dchi = _gather_units(wl, idx, got["dchi2"], False)
    tol_f = sbgpu.flux_tolerance(sub, ref["flux"], 1, False)
    assert np.all(np.abs(g_flux - ref["flux"]) <= tol_f)
    tol_d = sbgpu.grad_tolerance(sub, ref, sub.theta, 1, False)
    assert np.all(np.abs(g_dflux - ref["dflux"]) <= tol_d)
    tol_g = sbgpu.dchi2_tolerance(sub, ref, tol_f, tol_d, 1, False)
    assert np.all(np.abs(g_dchi - ref["dchi2"]) <= tol_g)
    assert np.all(np.isfinite(got["dchi2"]))


def test_full_size_config5_host_buffer_call_in_chunks(cuda_device):
    """sb_chi2_host on the whole of config 5 (195 MB of pinned host buffers: eight chunks staged with
    copy / compute overlap, the call bench.py's `e2e` times), sampled units against the oracle."""
    import torch

    import paper_2504_08081_b200 as sb

    wl = workloads.make_workload(5)
    idx = _sample_indices(wl.n_sn, 200, 91)
    sub = _attach_sampled(wl, idx)
    ref = oracle.run_workload(sub, want_flux=True, want_chi2=True)
    model, bands = sbgpu.load_handles(wl)
    ft = torch.float32

    def pin(a, dtype=ft):
        return torch.as_tensor(np.ascontiguousarray(a)).to(dtype).contiguous().pin_memory()

    o_flux = torch.full((wl.n_evals,), float("nan"), dtype=ft).pin_memory()
    o_chi = torch.full((wl.n_sn,), float("nan"), dtype=ft).pin_memory()
    sb.sb_chi2_host(model, bands, dtype=sb.SB_F32, n_sn=wl.n_sn, n_samples=1, n_obs_total=wl.n_obs_total,
                    obs_offset=pin(wl.obs_offset, torch.int32), time=pin(wl.time), band=pin(wl.band, torch.int32),
                    zp=pin(wl.zp), z=pin(wl.z), x0=pin(wl.theta["x0"]), x1=pin(wl.theta["x1"]), c=pin(wl.theta["c"]),
                    t0=pin(wl.theta["t0"]), flux=pin(wl.flux), fluxerr=pin(wl.fluxerr), out_chi2=o_chi, out_flux=o_flux)
    assert sb.last_launch_count() >= 6 and sb.last_form() == "tiled"  # several chunks, three kernels each
    got_flux, got_chi = o_flux.double().numpy(), o_chi.double().numpy()
    assert np.all(np.isfinite(got_flux)) and np.all(np.isfinite(got_chi))  # every chunk wrote its outputs
    tol = sbgpu.flux_tolerance(sub, ref["flux"], 1, False)
    err = np.abs(_gather_units(wl, idx, got_flux, True) - ref["flux"])
    assert np.all(err <= tol), f"worst flux err/tol {np.max(err / np.maximum(tol, 1e-300)):.3g}"
    tolc = sbgpu.chi2_tolerance(sub, ref["flux"], tol, 1, False)
    assert np.all(np.abs(_gather_units(wl, idx, got_chi, False) - ref["chi2"]) <= tolc)


def test_full_size_config5_nonuniform_band_grids(cuda_device):
    """The whole of config 5 with band grids jittered by +-30 % of the step (bench.py --band-jitter 0.3):
    the node-weight kernel's NU variant on sampled units against the oracle and on ALL units against the
    direct kernel."""
    wl = workloads.make_workload(5, band_jitter=0.3)
    idx = _sample_indices(wl.n_sn, 600, 123)
    sub = _attach_sampled(wl, idx)
    ref = oracle.run_workload(sub, want_flux=True, want_chi2=True)
    got = sbgpu.run_gpu(wl, mode="chi2")
    assert got["form"] == "tiled"
    tol = sbgpu.flux_tolerance(sub, ref["flux"], 1, False)
    err = np.abs(_gather_units(wl, idx, got["flux"], True) - ref["flux"])
    assert np.all(err <= tol), f"worst flux err/tol {np.max(err / np.maximum(tol, 1e-300)):.3g}"
    tolc = sbgpu.chi2_tolerance(sub, ref["flux"], tol, 1, False)
    assert np.all(np.abs(_gather_units(wl, idx, got["chi2"], False) - ref["chi2"]) <= tolc)
    direct = sbgpu.run_gpu(wl, mode="chi2", form="direct")
    peak = sbgpu.unit_peaks(wl, direct["flux"], 1)
    tol_all = 2.0 * (1e-5 * np.abs(direct["flux"]) + 1e-9 * peak)
    err_all = np.abs(got["flux"] - direct["flux"])
    assert np.all(err_all <= tol_all), f"tiled vs direct worst ratio {np.max(err_all / np.maximum(tol_all, 1e-300)):.3g}"
