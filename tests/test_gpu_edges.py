"""-m gpu edge cases: empty and ragged inputs, degenerate grids (every cell a border cell),
out-of-grid phases and bands, bad band indices, multi-tile rows, non-uniform band grids, a colour
law of maximum degree, scale invariance (P17) and the closed form P1 on the GPU."""
import numpy as np
import pytest

import oracle
import workloads
import sbgpu

pytestmark = pytest.mark.gpu

HC = 6.62607015e-27 * 2.99792458e18


def custom_workload(model, bands, obs_offset, time, band, z, theta, zp=25.0, n_samples=1):
    n_sn = len(z)
    n_tot = int(obs_offset[-1])
    f32 = lambda a: np.asarray(a, dtype=np.float64).astype(np.float32)
    wl = workloads.Workload(
        config=0, name="custom", model=model, bands=bands, n_sn=n_sn, n_samples=n_samples,
        obs_offset=np.asarray(obs_offset, dtype=np.int32), time=f32(time), band=np.asarray(band, dtype=np.int32),
        zp=f32(np.full(n_tot, zp)), z=f32(z), theta_true={k: f32(v) for k, v in theta.items()},
        theta={k: f32(v) for k, v in theta.items()}, noise=np.zeros(n_tot))
    return wl


def small_model(n_phase=3, n_wave=3, seed=1, w0=3000.0, dw=10.0, n_cl=5):
    rng = np.random.default_rng(seed)
    phase = -1.0 + np.arange(n_phase, dtype=np.float64)
    wave = w0 + dw * np.arange(n_wave, dtype=np.float64)
    cl = np.array([0.0, 0.8, -0.2, 0.05, -0.01, 0.002, -0.0003, 0.00004])[:n_cl]
    return {"phase": phase, "wave": wave, "m0": rng.uniform(0.5, 1.5, (n_phase, n_wave)),
            "m1": 0.1 * rng.standard_normal((n_phase, n_wave)), "cl_coef": cl, "cl_wave_b": 4302.57,
            "cl_wave_v": 5428.55, "cl_lo": 2800.0, "cl_hi": 7000.0}


def compare(wl, fp64, mode="grad"):
    ref = oracle.run_workload(wl, want_flux=True, want_dflux=True)
    got = sbgpu.run_gpu(wl, mode=mode, fp64=fp64, with_data=False)
    ns = wl.n_samples
    fin = np.isfinite(ref["flux"])
    tol = sbgpu.flux_tolerance(wl, np.where(fin, ref["flux"], 0.0), ns, fp64)
    assert np.array_equal(np.isnan(got["flux"]), np.isnan(ref["flux"]))
    assert np.all(np.abs(got["flux"] - ref["flux"])[fin] <= tol[fin])
    if mode == "grad":
        ref_f = {"flux": np.where(fin, ref["flux"], 0.0), "dflux": np.where(fin[:, None], ref["dflux"], 0.0)}
        tol_d = sbgpu.grad_tolerance(wl, ref_f, wl.theta, ns, fp64)
        assert np.all(np.abs(got["dflux"] - ref["dflux"])[fin] <= tol_d[fin])
    return got, ref


@pytest.mark.parametrize("fp64", [False, True])
@pytest.mark.parametrize("n_phase,n_wave", [(2, 2), (3, 3), (4, 5), (6, 6)])
def test_tiny_grids_border_cells(cuda_device, fp64, n_phase, n_wave):
    md = small_model(n_phase, n_wave, w0=3000.0, dw=40.0)
    span = 40.0 * (n_wave - 1)
    w = np.linspace(3000.0 - 20.0, 3000.0 + span + 20.0, 57) * 1.1  # straddles both grid edges at z = 0.1
    bd = workloads.generators.pack_bands([(w, np.linspace(0.2, 1.0, 57))])
    n = 40
    rng = np.random.default_rng(5)
    t = rng.uniform(-1.4, n_phase - 1.6, n)  # some phases outside the grid
    wl = custom_workload(md, bd, [0, n], t, np.zeros(n), [0.1],
                         {"x0": [1e-5], "x1": [0.7], "c": [0.1], "t0": [0.05]})
    compare(wl, fp64)


@pytest.mark.parametrize("fp64", [False, True])
def test_empty_and_degenerate_batches(cuda_device, fp64):
    import torch

    import paper_2504_08081_b200 as sb

    wl = workloads.make_workload(1)
    model, bands = sbgpu.load_handles(wl)
    ft = torch.float64 if fp64 else torch.float32
    dev = torch.device("cuda:0")
    z = torch.zeros(0, dtype=ft, device=dev)
    out = torch.zeros(0, dtype=ft, device=dev)
    # n_sn = 0: a no-op that succeeds and launches nothing
    sb.sb_bandflux(model, bands, dtype=sb.SB_F64 if fp64 else sb.SB_F32, n_sn=0, n_samples=1, n_obs_total=0,
                   obs_offset=torch.zeros(1, dtype=torch.int32, device=dev), time=out, band=torch.zeros(0, dtype=torch.int32, device=dev),
                   zp=None, z=z, x0=z, x1=z, c=z, t0=z, out_flux=out)
    assert sb.last_launch_count() == 0
    # supernovae with zero observations between others: chi2 = 0 for them
    md = wl.model
    wl2 = custom_workload(md, wl.bands, [0, 0, 5, 5, 9], np.linspace(-5, 30, 9), np.arange(9) % 4,
                          [0.1, 0.2, 0.3, 0.4], {"x0": [1e-5] * 4, "x1": [0.1] * 4, "c": [0.0] * 4, "t0": [0.0] * 4})
    ref = oracle.run_workload(wl2, want_flux=True)["flux"]
    workloads.attach_data(wl2, ref)
    got = sbgpu.run_gpu(wl2, mode="chi2", fp64=fp64)
    refc = oracle.run_workload(wl2, want_flux=True, want_chi2=True)
    assert got["chi2"][0] == 0.0 and got["chi2"][2] == 0.0
    tol2 = sbgpu.flux_tolerance(wl2, refc["flux"], 1, fp64)
    assert np.all(np.abs(got["chi2"] - refc["chi2"]) <= sbgpu.chi2_tolerance(wl2, refc["flux"], tol2, 1, fp64))
    assert np.all(np.abs(got["flux"] - refc["flux"]) <= tol2)


@pytest.mark.parametrize("fp64", [False, True])
def test_out_of_grid_and_bad_band(cuda_device, fp64):
    wl0 = workloads.make_workload(1)
    n = 12
    t = np.array([-30.0, -21.1, -20.0, 0.0, 49.9, 50.0, 52.5, 80.0, 1.0, 2.0, 3.0, 4.0])
    band = np.array([0, 1, 2, 3, 0, 1, 2, 3, -1, 4, 0, 99])
    wl = custom_workload(wl0.model, wl0.bands, [0, n], t, band, [0.0],
                         {"x0": [1e-5], "x1": [0.3], "c": [0.02], "t0": [0.0]})
    got, ref = compare(wl, fp64)
    assert np.isnan(got["flux"][8]) and np.isnan(got["flux"][9]) and np.isnan(got["flux"][11])
    assert got["flux"][0] == 0.0 and got["flux"][7] == 0.0 and got["flux"][6] == 0.0
    assert got["flux"][2] > 0.0 and got["flux"][5] > 0.0  # closed interval in phase
    # band entirely redward of the model grid at z = 0: zero
    w = 11500.0 + 5.0 * np.arange(41)
    bd = workloads.generators.pack_bands([(w, np.ones(41))])
    wl = custom_workload(wl0.model, bd, [0, 2], [0.0, 1.0], [0, 0], [0.0], {"x0": [1e-5], "x1": [0.3], "c": [0.02], "t0": [0.0]})
    got, _ = compare(wl, fp64)
    assert np.all(got["flux"] == 0.0) and np.all(got["dflux"] == 0.0)


@pytest.mark.parametrize("fp64", [False, True])
def test_multi_tile_rows_and_nonuniform_band(cuda_device, fp64):
    """A 1 A model grid makes one band span ~5000 cells: several passes of the warp's row buffer."""
    rng = np.random.default_rng(3)
    n_wave = 6001
    phase = -5.0 + np.arange(12, dtype=np.float64)
    wave = 3000.0 + 1.0 * np.arange(n_wave)
    lam = wave[None, :]
    m0 = (1.0 + 0.3 * np.sin(lam / 37.0)) * np.exp(-0.5 * (phase[:, None] / 6.0) ** 2)
    md = {"phase": phase, "wave": wave, "m0": m0, "m1": 0.1 * m0 * np.cos(lam / 91.0 + phase[:, None]),
          "cl_coef": np.array([0.0, 0.8, -0.2, 0.05, -0.01]), "cl_wave_b": 4302.57, "cl_wave_v": 5428.55,
          "cl_lo": 2800.0, "cl_hi": 7000.0}
    w_a = np.sort(rng.uniform(3500.0, 8700.0, 900))  # non-uniform grid
    w_a[0], w_a[-1] = 3500.0, 8700.0
    w_b = 2900.0 + 2.5 * np.arange(2600)  # straddles the blue edge, 2600 samples
    bd = workloads.generators.pack_bands([(w_a, np.exp(-0.5 * ((w_a - 6000.0) / 900.0) ** 2)),
                                          (w_b, np.full(w_b.size, 0.7))])
    n = 24
    wl = custom_workload(md, bd, [0, n // 2, n], rng.uniform(-4.0, 5.5, n), np.arange(n) % 2, [0.0, 0.31],
                         {"x0": [1e-5, 3e-5], "x1": [0.7, -1.2], "c": [0.1, -0.2], "t0": [0.05, -0.3]})
    compare(wl, fp64)
    compare(wl, fp64, mode="flux")


@pytest.mark.parametrize("fp64", [False, True])
def test_degree7_colour_law(cuda_device, fp64):
    wl0 = workloads.make_workload(1)
    md = dict(wl0.model)
    md["cl_coef"] = np.array([0.01, 0.8, -0.2, 0.05, -0.01, 0.002, -0.0003, 0.00002])
    wl = custom_workload(md, wl0.bands, wl0.obs_offset, wl0.time, wl0.band, [0.05],
                         {"x0": [1e-5], "x1": [0.5], "c": [0.25], "t0": [0.0]})
    compare(wl, fp64)


def test_p1_closed_form_on_gpu(cuda_device):
    K, x0 = 3.25, 2.0e-5
    phase = -5.0 + np.arange(11.0)
    wave = 3000.0 + 10.0 * np.arange(101)
    md = {"phase": phase, "wave": wave, "m0": np.full((11, 101), K), "m1": np.zeros((11, 101)),
          "cl_coef": np.array([0.0, 1.0, -0.2]), "cl_wave_b": 4302.57, "cl_wave_v": 5428.55, "cl_lo": 2800.0, "cl_hi": 7000.0}
    la, lb = 3700.0, 3900.0
    w = la + 5.0 * np.arange(41)
    bd = workloads.generators.pack_bands([(w, np.ones(41))])
    wl = custom_workload(md, bd, [0, 3], [0.3, -2.2, 3.9], [0, 0, 0], [0.05],
                         {"x0": [x0], "x1": [0.7], "c": [0.0], "t0": [0.1]})
    want = float(np.float32(x0)) * K * (lb * lb - la * la) / (2.0 * HC)  # x0 as the fp32 value both sides get
    for fp64, tol in ((False, 1e-6), (True, 1e-13)):
        got = sbgpu.run_gpu(wl, mode="flux", fp64=fp64, use_zp=False)["flux"]
        assert np.all(np.abs(got - want) <= tol * want)


@pytest.mark.parametrize("kappa", [1e-12, 1e6])
def test_p17_scale_invariance_fp32(cuda_device, kappa):
    wl = workloads.make_workload(2, n_sn=16)
    a = sbgpu.run_gpu(wl, mode="flux")["flux"]
    md = dict(wl.model)
    md["m0"], md["m1"] = wl.model["m0"] * kappa, wl.model["m1"] * kappa
    th = {k: v.copy() for k, v in wl.theta.items()}
    th["x0"] = (th["x0"].astype(np.float64) / kappa).astype(np.float32)
    wl2 = custom_workload(md, wl.bands, wl.obs_offset, wl.time, wl.band, wl.z, th)
    b = sbgpu.run_gpu(wl2, mode="flux")["flux"]
    x0_ratio = th["x0"].astype(np.float64) * kappa / wl.theta["x0"].astype(np.float64)  # fp32 rounding of x0/kappa
    b = b / np.repeat(x0_ratio, np.diff(wl.obs_offset))
    assert np.all(np.abs(a - b) <= 2e-6 * np.abs(a) + 1e-9 * np.max(np.abs(a)))


@pytest.mark.parametrize("config", [1, 5])
def test_zpab_of_the_loader_equals_the_oracle(cuda_device, config):
    """a0 / reading G7: ZPAB_b as sb_load_bandpasses computes it at load (fp64 host arithmetic, folded
    weights) against the oracle's literal trapezoid of the AB spectrum through the band, for every band of
    configs 1 and 5 (optical and NIR), and on jittered (non-uniform) grids of the same bands."""
    for jitter in (0.0, 0.3):
        wl = workloads.make_workload(config, **({"n_sn": 4} if config == 5 else {}))
        if jitter:
            wl.bands = workloads.jitter_band_grids(wl.bands, jitter)
        _, bands = sbgpu.load_handles(wl)
        ob = oracle.Bands.from_dict(wl.bands)
        n_bands = len(wl.bands["offset"]) - 1
        assert bands.n_bands == n_bands
        for b in range(n_bands):
            want = ob.zpab(b)
            assert want > 0 and abs(bands.zpab(b) - want) <= 1e-14 * want, (config, jitter, b)
        assert np.isnan(bands.zpab(n_bands)) and np.isnan(bands.zpab(-1))
