"""-m gpu edge cases of the grouped / tiled formulations (csrc/sb_hoist.cuh, csrc/sb_nw.cuh), each
against the fp64 oracle and in every formulation that applies: windows wider than one 512-node
segment of the node-weight array, a unit with more observations than one round holds (the unit is
split over rounds and its chi^2 carried), empty units inside a group, groups that mix very different
redshifts (union node window much wider than any item's), bands that leave the model grid for
part of a group, a single band, and phases outside the grid."""
import numpy as np
import pytest

import oracle
import sbgpu
import workloads
from test_gpu_edges import custom_workload

pytestmark = pytest.mark.gpu

CL = {"cl_coef": np.array([0.0, 0.8, -0.2, 0.05, -0.01]), "cl_wave_b": 4302.57, "cl_wave_v": 5428.55,
      "cl_lo": 2800.0, "cl_hi": 7000.0}


def smooth_model(n_phase, wave, seed=0):
    phase = -6.0 + np.arange(n_phase, dtype=np.float64)
    lam = wave[None, :]
    taper = np.clip((lam - wave[0]) / 200.0, 0, 1) * np.clip((wave[-1] - lam) / 200.0, 0, 1)
    m0 = (1.0 + 0.3 * np.sin(lam / 137.0 + seed)) * np.exp(-0.5 * (phase[:, None] / 7.0) ** 2) * taper
    m1 = 0.1 * m0 * np.cos(lam / 291.0 + 0.3 * phase[:, None])
    return dict(phase=phase, wave=wave, m0=m0, m1=m1, **CL)


def attach(wl):
    true = oracle.run_workload(wl, theta={k: v.copy() for k, v in wl.theta_true.items()}, want_flux=True)["flux"]
    rng = np.random.default_rng(9)
    wl.noise = rng.standard_normal(wl.n_obs_total)
    workloads.attach_data(wl, np.where(np.isfinite(true), true, 0.0))
    return wl


def check_all_forms(wl, forms=("tiled", "grouped", "direct"), grad_forms=("tiled", "direct")):
    ns = wl.n_samples
    ref = oracle.run_workload(wl, want_flux=True, want_chi2=True, want_dflux=True, want_dchi2=True)
    fin = np.isfinite(ref["flux"])
    ref0 = {"flux": np.where(fin, ref["flux"], 0.0), "dflux": np.where(fin[:, None], ref["dflux"], 0.0)}
    tol = sbgpu.flux_tolerance(wl, ref0["flux"], ns, False)
    tolc = sbgpu.chi2_tolerance(wl, ref0["flux"], tol, ns, False)
    tol_d = sbgpu.grad_tolerance(wl, ref0, wl.theta, ns, False)
    okc = np.isfinite(ref["chi2"])
    for form in forms:
        try:
            got = sbgpu.run_gpu(wl, mode="chi2", form=form)
        except Exception as exc:  # include/saltband.h: SB_ELIMIT when a demanded formulation does not apply
            assert form == "grouped" and "status -4" in str(exc), (form, exc)  # model wider than its table
            continue
        assert got["form"] == form
        assert np.array_equal(np.isnan(got["flux"]), ~fin), form
        err = np.abs(got["flux"] - ref["flux"])[fin]
        assert np.all(err <= tol[fin]), (form, float(np.max(err / np.maximum(tol[fin], 1e-300))))
        assert np.all(np.abs(got["chi2"] - ref["chi2"])[okc] <= tolc[okc]), form
    for form in grad_forms:
        got = sbgpu.run_gpu(wl, mode="grad", form=form)
        assert got["form"] == form
        assert np.all(np.abs(got["flux"] - ref["flux"])[fin] <= tol[fin]), form
        errd = np.abs(got["dflux"] - ref["dflux"])[fin]
        assert np.all(errd <= tol_d[fin]), (form, np.max(errd / np.maximum(tol_d[fin], 1e-300), axis=0))
        tol_g = sbgpu.dchi2_tolerance(wl, {"flux": ref0["flux"], "dflux": ref0["dflux"]}, tol, tol_d, ns, False)
        assert np.all(np.abs(got["dchi2"] - ref["dchi2"])[okc] <= tol_g[okc]), form
        assert np.all(np.abs(got["chi2"] - ref["chi2"])[okc] <= tolc[okc]), form


def test_windows_wider_than_one_segment(cuda_device):
    """2 A model grid: a 3000 A band spans ~1400 nodes at z ~ 0.05 (three 512-node segments); the
    second band leaves the grid on the blue side for the high-redshift units of the same group."""
    wave = 3000.0 + 2.0 * np.arange(2501)  # 3000 .. 8000 A
    md = smooth_model(14, wave)
    w_a = 4000.0 + 5.0 * np.arange(601)    # 4000 .. 7000 A
    w_b = 3050.0 + 5.0 * np.arange(241)    # 3050 .. 4250 A: rest frame < 3000 A for z > 0.42
    bd = workloads.generators.pack_bands([(w_a, np.exp(-0.5 * ((w_a - 5500.0) / 700.0) ** 2)),
                                          (w_b, np.full(w_b.size, 0.6))])
    rng = np.random.default_rng(1)
    n_sn, n_obs = 9, 12
    z = np.array([0.05, 0.051, 0.30, 0.02, 0.5, 0.049, 0.31, 0.0, 0.8])
    th = {"x0": rng.uniform(1e-5, 3e-5, n_sn), "x1": rng.normal(size=n_sn), "c": 0.1 * rng.normal(size=n_sn),
          "t0": rng.uniform(-1, 1, n_sn)}
    wl = custom_workload(md, bd, np.arange(n_sn + 1) * n_obs, rng.uniform(-5.0, 6.5, n_sn * n_obs),
                         np.arange(n_sn * n_obs) % 2, z, th)
    check_all_forms(attach(wl))


def test_unit_larger_than_a_round_and_empty_units(cuda_device):
    """One supernova with 3500 observations (> 3072 per forward round, > 1536 per gradient round), two
    with none, the rest ragged: segments, chi^2 carry over rounds, empty units (chi^2 = 0)."""
    wl0 = workloads.make_workload(2, n_sn=8)
    rng = np.random.default_rng(2)
    counts = np.array([5, 0, 3500, 17, 0, 60, 1, 33])
    off = np.concatenate([[0], np.cumsum(counts)])
    n = int(off[-1])
    th = {k: v.astype(np.float64) for k, v in wl0.theta.items()}
    wl = custom_workload(wl0.model, wl0.bands, off, rng.uniform(-15.0, 45.0, n), rng.integers(0, 6, n),
                         wl0.z.astype(np.float64), th)
    wl = attach(wl)
    check_all_forms(wl)
    got = sbgpu.run_gpu(wl, mode="chi2", form="tiled")
    assert got["chi2"][1] == 0.0 and got["chi2"][4] == 0.0


@pytest.mark.parametrize("n_bands", [1, 3, 5])
def test_split_unit_with_odd_band_counts(cuda_device, n_bands):
    """A unit larger than a round (chi^2 and d chi^2 carried between rounds in fp64 shared memory) with an
    ODD number of (band, segment) items: the carry must stay 8-byte aligned whatever the item count
    (round-1 advisor finding).  Forward and gradient, node-weight kernel against the oracle."""
    wl0 = workloads.make_workload(2, n_sn=3)
    bd = wl0.bands
    sub = workloads.generators.pack_bands([(bd["wave"][bd["offset"][b]:bd["offset"][b + 1]],
                                            bd["trans"][bd["offset"][b]:bd["offset"][b + 1]]) for b in range(n_bands)])
    rng = np.random.default_rng(20 + n_bands)
    counts = np.array([3300, 7, 1700])
    off = np.concatenate([[0], np.cumsum(counts)])
    n = int(off[-1])
    th = {k: v.astype(np.float64) for k, v in wl0.theta.items()}
    wl = custom_workload(wl0.model, sub, off, rng.uniform(-15.0, 45.0, n), rng.integers(0, n_bands, n),
                         wl0.z.astype(np.float64), th)
    check_all_forms(attach(wl), forms=("tiled",), grad_forms=("tiled",))


def test_single_band_phases_outside_grid_and_samples_axis(cuda_device):
    """One band, several parameter samples per supernova (units of one object share observations),
    t0 pushed so that part of the phases fall outside the phase grid (zero flux, G3)."""
    wave = 2500.0 + 10.0 * np.arange(651)
    md = smooth_model(9, wave, seed=2)  # phases -6 .. +2 d
    w = 4500.0 + 5.0 * np.arange(301)
    bd = workloads.generators.pack_bands([(w, np.exp(-0.5 * ((w - 5250.0) / 300.0) ** 2))])
    rng = np.random.default_rng(4)
    n_sn, n_samples, n_obs = 3, 21, 37
    z = np.array([0.1, 0.45, 0.0])
    nu = n_sn * n_samples
    th = {"x0": rng.uniform(1e-5, 3e-5, nu), "x1": rng.normal(size=nu), "c": 0.1 * rng.normal(size=nu),
          "t0": rng.uniform(-4, 4, nu)}
    wl = custom_workload(md, bd, np.arange(n_sn + 1) * n_obs, rng.uniform(-9.0, 5.0, n_sn * n_obs),
                         np.zeros(n_sn * n_obs, dtype=int), z, th, n_samples=n_samples)
    wl.theta_true = {k: v.reshape(n_sn, n_samples)[:, 0].copy() for k, v in wl.theta.items()}
    wl = attach(wl)
    ref = oracle.run_workload(wl, want_flux=True)["flux"]
    assert 0.05 < np.mean(ref == 0.0) < 0.9  # the case does exercise out-of-grid phases
    check_all_forms(wl)


@pytest.mark.parametrize("seed", [11, 12, 13, 14, 15, 16])
def test_random_grids_band_steps_and_redshifts(cuda_device, seed):
    """Seeded random cases: model grid steps 2-25 A, band steps from a tenth of a model cell to
    three cells (cells with no band sample at all), 1-5 bands partly outside the grid, redshifts
    -0.05 .. 2, 1-40 units with 0-30 observations, 1-3 samples per supernova; every formulation."""
    rng = np.random.default_rng(seed)
    dw = float(rng.choice([2.0, 5.0, 10.0, 25.0]))
    n_wave = int(rng.integers(40, 900))
    wave = 2500.0 + dw * np.arange(n_wave)
    md = smooth_model(int(rng.integers(4, 12)), wave, seed=seed)
    bands = []
    for _ in range(int(rng.integers(1, 6))):
        h = dw * float(rng.choice([0.1, 0.37, 0.5, 1.0, 1.7, 3.0]))
        lo = float(rng.uniform(wave[0] - 400.0, wave[-1] * 1.5))
        n = int(rng.integers(5, 400))
        w = lo + h * np.arange(n)
        bands.append((w, 0.2 + 0.8 * np.exp(-0.5 * ((w - w.mean()) / (0.3 * (w[-1] - w[0]) + 1.0)) ** 2)))
    bd = workloads.generators.pack_bands(bands)
    n_sn, ns = int(rng.integers(1, 41)), int(rng.integers(1, 4))
    counts = rng.integers(0, 31, n_sn)
    off = np.concatenate([[0], np.cumsum(counts)])
    n = int(off[-1])
    nu = n_sn * ns
    z = rng.uniform(-0.05, 2.0, n_sn)
    th = {"x0": rng.uniform(1e-5, 3e-5, nu), "x1": rng.normal(size=nu), "c": 0.15 * rng.normal(size=nu),
          "t0": rng.uniform(-2, 2, nu)}
    phase = md["phase"]
    wl = custom_workload(md, bd, off, rng.uniform(phase[0] - 2.0, (phase[-1] + 2.0) * 1.5, n),
                         rng.integers(0, len(bands), n), z, th, n_samples=ns)
    wl.theta_true = {k: v.reshape(n_sn, ns)[:, 0].copy() for k, v in wl.theta.items()}
    if n == 0:
        return
    check_all_forms(attach(wl))


def test_groups_of_exactly_32_units(cuda_device):
    """148 x 32 supernovae: every CTA's group holds exactly 32 units (a full warp of segment lanes in the
    round builder; the host-buffer calls cut their chunks to such multiples) -- forward and gradient."""
    import torch

    n_sm = torch.cuda.get_device_properties(0).multi_processor_count
    wl = workloads.make_workload(2, n_sn=32 * n_sm)
    true = oracle.run_workload(wl, theta={k: v.copy() for k, v in wl.theta_true.items()})["flux"]
    workloads.attach_data(wl, true)
    ref = oracle.run_workload(wl, want_flux=True, want_chi2=True)
    got = sbgpu.run_gpu(wl, mode="chi2", form="tiled")
    tol = sbgpu.flux_tolerance(wl, ref["flux"], 1, False)
    assert np.all(np.abs(got["flux"] - ref["flux"]) <= tol)
    assert np.all(np.abs(got["chi2"] - ref["chi2"]) <= sbgpu.chi2_tolerance(wl, ref["flux"], tol, 1, False))
    half = workloads.subset(wl, np.arange(16 * n_sm))  # gradient rounds hold 16 units
    refg = oracle.run_workload(half, want_flux=True, want_dflux=True)
    gotg = sbgpu.run_gpu(half, mode="grad", form="tiled", with_data=False)
    assert np.all(np.abs(gotg["dflux"] - refg["dflux"]) <= sbgpu.grad_tolerance(half, refg, half.theta, 1, False))
