"""-m gpu parity tests: the CUDA path (through the C ABI) against the fp64 oracle, element by
element, on the same seeded inputs (BASELINE.json configs, reduced to sizes the oracle finishes in
seconds but spanning many CTAs, warps, tiles and ragged tails), plus edge cases.
Tolerances: DESIGN.md reading G13 (tests/sbgpu.py); fp32 1e-5 rel + 1e-9 peak, fp64 1e-12."""
import numpy as np
import pytest

import oracle
import workloads
import sbgpu

pytestmark = pytest.mark.gpu


def theta_true_rep(wl):
    return {k: v.copy() for k, v in wl.theta_true.items()}


def prepare(config, **kw):
    """Workload with photometry attached from the ORACLE's flux at theta_true."""
    wl = workloads.make_workload(config, **kw)
    ref_true = oracle.run_workload(wl, theta=theta_true_rep(wl), want_flux=True)["flux"]
    workloads.attach_data(wl, ref_true)
    return wl


def oracle_all(wl, grad=False):
    return oracle.run_workload(wl, want_flux=True, want_chi2=True, want_dflux=grad, want_dchi2=grad)


def check_flux_chi2(wl, got, ref, fp64):
    ns = wl.n_samples
    tol = sbgpu.flux_tolerance(wl, ref["flux"], ns, fp64)
    err = np.abs(got["flux"] - ref["flux"])
    bad = np.nonzero(~(err <= tol))[0]
    assert bad.size == 0, f"{bad.size} flux mismatches, worst ratio {np.max(err / np.maximum(tol, 1e-300)):.3g}"
    if "chi2" in got:
        tolc = sbgpu.chi2_tolerance(wl, ref["flux"], tol, ns, fp64)
        errc = np.abs(got["chi2"] - ref["chi2"])
        assert np.all(errc <= tolc), f"chi2 worst ratio {np.max(errc / np.maximum(tolc, 1e-300)):.3g}"
    return float(np.max(err / np.maximum(tol, 1e-300)))


@pytest.mark.parametrize("fp64", [False, True])
def test_config1_full(cuda_device, fp64):
    wl = prepare(1)
    ref = oracle_all(wl)
    got = sbgpu.run_gpu(wl, mode="chi2", fp64=fp64)
    assert got["launches"] >= 1
    check_flux_chi2(wl, got, ref, fp64)
    only_flux = sbgpu.run_gpu(wl, mode="flux", fp64=fp64)
    assert np.array_equal(only_flux["flux"], got["flux"])


@pytest.mark.parametrize("fp64", [False, True])
def test_config2_full_and_ragged(cuda_device, fp64):
    wl = prepare(2)  # 1024 SN x 60 obs: full size
    ref = oracle_all(wl)
    got = sbgpu.run_gpu(wl, mode="chi2", fp64=fp64)
    check_flux_chi2(wl, got, ref, fp64)
    assert np.mean(ref["flux"] == 0.0) < 0.2
    wlr = prepare(2, n_sn=97, ragged=True)
    check_flux_chi2(wlr, sbgpu.run_gpu(wlr, mode="chi2", fp64=fp64), oracle_all(wlr), fp64)


@pytest.mark.parametrize("fp64", [False, True])
def test_config3_samples_axis(cuda_device, fp64):
    wl = prepare(3, n_samples=300)  # 1 SN x 300 samples x 50 obs
    ref = oracle_all(wl)
    got = sbgpu.run_gpu(wl, mode="chi2", fp64=fp64)
    check_flux_chi2(wl, got, ref, fp64)
    # chi2 only (no flux output), as the nested-sampling likelihood is called
    got2 = sbgpu.run_gpu(wl, mode="chi2", fp64=fp64, want_flux=False)
    assert np.array_equal(got2["chi2"], got["chi2"])


@pytest.mark.parametrize("fp64,form", [(False, None), (False, "direct"), (False, "tiled"), (True, None)])
def test_config4_forward_and_gradient(cuda_device, fp64, form):
    wl = prepare(4, n_sn=160)
    ref = oracle_all(wl, grad=True)
    got = sbgpu.run_gpu(wl, mode="grad", fp64=fp64, form=form)
    if form is not None:
        assert got["form"] == form
    ns = wl.n_samples
    check_flux_chi2(wl, got, ref, fp64)
    tol_f = sbgpu.flux_tolerance(wl, ref["flux"], ns, fp64)
    tol_d = sbgpu.grad_tolerance(wl, ref, wl.theta, ns, fp64)
    err = np.abs(got["dflux"] - ref["dflux"])
    assert np.all(err <= tol_d), f"dflux worst ratio per component {np.max(err / np.maximum(tol_d, 1e-300), axis=0)}"
    tol_g = sbgpu.dchi2_tolerance(wl, ref, tol_f, tol_d, ns, fp64)
    errg = np.abs(got["dchi2"] - ref["dchi2"])
    assert np.all(errg <= tol_g), f"dchi2 worst ratio {np.max(errg / np.maximum(tol_g, 1e-300), axis=0)}"
    # the grad kernel's forward equals the forward kernel's within tolerance
    fwd = sbgpu.run_gpu(wl, mode="chi2", fp64=fp64)
    assert np.all(np.abs(fwd["flux"] - got["flux"]) <= 2 * tol_f)


def test_config4_gpu_gradient_vs_oracle_central_differences(cuda_device):
    """BASELINE.json configs[3]: analytic gradient against ORACLE central differences, step 1e-6 rel."""
    wl = prepare(4, n_sn=24)
    ns = wl.n_samples
    base = oracle.run_workload(wl, want_flux=True, want_dflux=True)
    for fp64 in (False, True):
        got = sbgpu.run_gpu(wl, mode="grad", fp64=fp64, with_data=False)
        tol_d = sbgpu.grad_tolerance(wl, base, wl.theta, ns, fp64)
        peak = sbgpu.unit_peaks(wl, base["flux"], ns)
        for q, key in enumerate(("x0", "x1", "c", "t0")):
            th = wl.theta[key].astype(np.float64)
            h = 1e-6 * (np.abs(th) if key == "x0" else np.maximum(np.abs(th), 1.0))
            up = {k: v.astype(np.float64).copy() for k, v in wl.theta.items()}
            dn = {k: v.astype(np.float64).copy() for k, v in wl.theta.items()}
            up[key] = th + h
            dn[key] = th - h
            fu = oracle.run_workload(wl, theta=up)["flux"]
            fd = oracle.run_workload(wl, theta=dn)["flux"]
            hh = np.repeat(h, np.diff(wl.obs_offset))
            fdiff = (fu - fd) / (2.0 * hh)
            scale = np.repeat(np.maximum(np.abs(th), 1.0) if key != "x0" else np.abs(th), np.diff(wl.obs_offset))
            tol = tol_d[:, q] + 1e-6 * np.maximum(np.abs(base["dflux"][:, q]), peak / scale)
            err = np.abs(got["dflux"][:, q] - fdiff)
            assert np.all(err <= tol), (key, fp64, float(np.max(err / tol)))


@pytest.mark.parametrize("fp64", [False, True])
def test_config5_nir_grid(cuda_device, fp64):
    wl = prepare(5, n_sn=300)  # 24000 evals on the 71 x 1801 grid, 10 bands up to 961 samples
    ref = oracle_all(wl)
    got = sbgpu.run_gpu(wl, mode="chi2", fp64=fp64)
    check_flux_chi2(wl, got, ref, fp64)


def test_chi2_is_deterministic(cuda_device):
    wl = prepare(2, n_sn=200)
    a = sbgpu.run_gpu(wl, mode="chi2")
    b = sbgpu.run_gpu(wl, mode="chi2")
    assert np.array_equal(a["chi2"], b["chi2"]) and np.array_equal(a["flux"], b["flux"])


def test_no_zero_point_is_raw_photon_flux(cuda_device):
    wl = prepare(1)
    got = sbgpu.run_gpu(wl, mode="flux", use_zp=False)
    m, b = oracle.Model.from_dict(wl.model), oracle.Bands.from_dict(wl.bands)
    th = wl.theta
    want = np.array([oracle.eval_one(m, b, float(wl.z[0]), float(wl.time[i]), int(wl.band[i]), None,
                                     float(th["x0"][0]), float(th["x1"][0]), float(th["c"][0]), float(th["t0"][0]))
                     for i in range(wl.n_obs_total)])
    assert np.all(np.abs(got["flux"] - want) <= 1e-5 * np.abs(want) + 1e-9 * np.max(np.abs(want)))


@pytest.mark.parametrize("form", ["direct", "grouped", "tiled"])
@pytest.mark.parametrize("config,kw", [(2, {"n_sn": 257, "ragged": True}), (3, {"n_samples": 200}), (5, {"n_sn": 200})])
def test_each_formulation_against_oracle(cuda_device, form, config, kw):
    """include/saltband.h SB_FORM_*: the per-evaluation kernel and the band-grouped kernel are both
    exact re-associations of the same sums; each is checked against the oracle on its own (fp32)."""
    wl = prepare(config, **kw)
    ref = oracle_all(wl)
    got = sbgpu.run_gpu(wl, mode="chi2", form=form)
    # sort kernel (small batch; not needed for a single supernova in the tiled form) + main
    assert got["launches"] == (1 if form == "direct" or (form == "tiled" and wl.n_sn == 1) else 2) and got["form"] == form
    check_flux_chi2(wl, got, ref, False)


def test_gradient_formulations_on_samples_axis_and_ragged_units(cuda_device):
    """sb_bandflux_grad in the tiled formulation where units share a supernova (config 3 shape: the
    group of a CTA is 16 parameter samples of one object) and where units are ragged (config 2 shape)."""
    for config, kw in ((3, {"n_samples": 150}), (2, {"n_sn": 133, "ragged": True}), (5, {"n_sn": 150})):
        wl = prepare(config, **kw)
        ref = oracle_all(wl, grad=True)
        ns = wl.n_samples
        for form in ("tiled", "direct"):
            got = sbgpu.run_gpu(wl, mode="grad", form=form)
            assert got["form"] == form
            check_flux_chi2(wl, got, ref, False)
            tol_f = sbgpu.flux_tolerance(wl, ref["flux"], ns, False)
            tol_d = sbgpu.grad_tolerance(wl, ref, wl.theta, ns, False)
            err = np.abs(got["dflux"] - ref["dflux"])
            assert np.all(err <= tol_d), (config, form, np.max(err / np.maximum(tol_d, 1e-300), axis=0))
            tol_g = sbgpu.dchi2_tolerance(wl, ref, tol_f, tol_d, ns, False)
            errg = np.abs(got["dchi2"] - ref["dchi2"])
            assert np.all(errg <= tol_g), (config, form, np.max(errg / np.maximum(tol_g, 1e-300), axis=0))


@pytest.mark.parametrize("fp64", [False, True])
def test_host_buffer_calls_equal_device_calls(cuda_device, fp64):
    """include/saltband.h sb_chi2_host / sb_bandflux_grad_host: staging of HOST buffers (pinned and
    pageable) through the library's device buffers; a workload that fits one chunk gives bit-identical
    results to the device calls, and matches the oracle.  (Several chunks: test_gpu_fullsize.py.)"""
    import torch

    import paper_2504_08081_b200 as sb

    wl = prepare(2, n_sn=700, ragged=True)
    ref = oracle_all(wl, grad=True)
    dev = sbgpu.run_gpu(wl, mode="grad", fp64=fp64)
    ft = torch.float64 if fp64 else torch.float32
    model, bands = sbgpu.load_handles(wl)

    def host(a, dtype=ft, pin=True):
        t = torch.as_tensor(np.ascontiguousarray(np.asarray(a, dtype=np.float64))).to(dtype).contiguous()
        return t.pin_memory() if pin else t

    n_tot, n_units = wl.n_obs_total, wl.n_sn * wl.n_samples
    for pin in (True, False):
        common = dict(dtype=sb.SB_F64 if fp64 else sb.SB_F32, n_sn=wl.n_sn, n_samples=wl.n_samples, n_obs_total=n_tot,
                      obs_offset=host(wl.obs_offset, torch.int32, pin), time=host(wl.time, ft, pin),
                      band=host(wl.band, torch.int32, pin), zp=host(wl.zp, ft, pin), z=host(wl.z, ft, pin),
                      x0=host(wl.theta["x0"], ft, pin), x1=host(wl.theta["x1"], ft, pin), c=host(wl.theta["c"], ft, pin),
                      t0=host(wl.theta["t0"], ft, pin))
        o_flux, o_dflux = torch.full((n_tot,), float("nan"), dtype=ft), torch.full((n_tot * 4,), float("nan"), dtype=ft)
        o_chi, o_dchi = torch.full((n_units,), float("nan"), dtype=ft), torch.full((n_units * 4,), float("nan"), dtype=ft)
        sb.sb_bandflux_grad_host(model, bands, flux=host(wl.flux, ft, pin), fluxerr=host(wl.fluxerr, ft, pin),
                                 out_flux=o_flux, out_dflux=o_dflux, out_chi2=o_chi, out_dchi2=o_dchi, **common)
        assert sb.last_launch_count() >= 1
        assert np.array_equal(o_flux.double().numpy(), dev["flux"])
        assert np.array_equal(o_dflux.double().numpy().reshape(-1, 4), dev["dflux"])
        assert np.array_equal(o_chi.double().numpy(), dev["chi2"])
        assert np.array_equal(o_dchi.double().numpy().reshape(-1, 4), dev["dchi2"])
        o_chi2 = torch.full((n_units,), float("nan"), dtype=ft)
        sb.sb_chi2_host(model, bands, flux=host(wl.flux, ft, pin), fluxerr=host(wl.fluxerr, ft, pin), out_chi2=o_chi2,
                        **common)
        tol = sbgpu.flux_tolerance(wl, ref["flux"], 1, fp64)
        tolc = sbgpu.chi2_tolerance(wl, ref["flux"], tol, 1, fp64)
        assert np.all(np.abs(o_chi2.double().numpy() - ref["chi2"]) <= tolc)
    check_flux_chi2(wl, dev, ref, fp64)


def test_host_buffer_call_chunks_with_samples_axis(cuda_device):
    """sb_chi2_host with several parameter samples per supernova and several chunks (the flux output
    of one supernova is 0.9 MB, so the 24 MB chunk target cuts 90 supernovae into four chunks).  In
    fp64 the library runs the per-evaluation kernel, whose results do not depend on how units are
    grouped: the chunked host call must equal the whole-batch device call bit for bit (flux) and to
    rounding of the per-unit sum (chi^2)."""
    import torch

    import paper_2504_08081_b200 as sb

    wl = workloads.make_workload(2, n_sn=90, ragged=True)
    ns = 2000
    rng = np.random.default_rng(17)
    nu = wl.n_sn * ns
    th = {"x0": np.repeat(wl.theta["x0"], ns) * rng.uniform(0.8, 1.2, nu), "x1": rng.normal(size=nu),
          "c": 0.1 * rng.normal(size=nu), "t0": rng.uniform(-3, 3, nu)}
    th = {k: v.astype(np.float32).astype(np.float64) for k, v in th.items()}
    wl.flux = (1e-3 * wl.noise).astype(np.float32)
    wl.fluxerr = np.full(wl.n_obs_total, 1e-3, dtype=np.float32)
    dev = sbgpu.run_gpu(wl, mode="chi2", fp64=True, theta=th)
    model, bands = sbgpu.load_handles(wl)
    ft = torch.float64

    def host(a, dtype=ft):
        return torch.as_tensor(np.ascontiguousarray(np.asarray(a, dtype=np.float64))).to(dtype).contiguous().pin_memory()

    n_tot = wl.n_obs_total
    o_flux = torch.full((n_tot * ns,), float("nan"), dtype=ft).pin_memory()
    o_chi = torch.full((nu,), float("nan"), dtype=ft).pin_memory()
    sb.sb_chi2_host(model, bands, dtype=sb.SB_F64, n_sn=wl.n_sn, n_samples=ns, n_obs_total=n_tot,
                    obs_offset=host(wl.obs_offset, torch.int32), time=host(wl.time), band=host(wl.band, torch.int32),
                    zp=host(wl.zp), z=host(wl.z), x0=host(th["x0"]), x1=host(th["x1"]), c=host(th["c"]),
                    t0=host(th["t0"]), flux=host(wl.flux), fluxerr=host(wl.fluxerr), out_chi2=o_chi, out_flux=o_flux)
    assert sb.last_launch_count() >= 3  # one direct-kernel launch per chunk
    assert np.array_equal(o_flux.numpy(), dev["flux"])
    # chi^2: the partial sums of a unit follow the kernel's evaluation chunks, which depend on the batch
    assert np.all(np.abs(o_chi.numpy() - dev["chi2"]) <= 1e-13 * np.abs(dev["chi2"]))
