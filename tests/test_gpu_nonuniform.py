"""-m gpu: non-uniformly sampled band grids (tabulated filters; reading G8: the band's own grid,
general trapezoid weights) on the node-weight kernel -- the NU variant of csrc/sb_nw.cuh, which reads each
sample's offset from the band's mean-step grid and finds the samples of a model cell by a local search.
Element-by-element against the oracle, forward and gradient, with and without a pack, and against the
direct kernel; grids: 5 A steps jittered by +-30 % (bounded offsets), and piecewise steps 5 / 10 / 25 A
(offsets of many steps: the search runs long but must stay exact)."""
import numpy as np
import pytest

import oracle
import sbgpu
import workloads

pytestmark = pytest.mark.gpu


def _prepare(wl):
    true = oracle.run_workload(wl, theta={k: v.copy() for k, v in wl.theta_true.items()})["flux"]
    workloads.attach_data(wl, true)
    return wl


def _check(wl, got, ref, grad):
    tol = sbgpu.flux_tolerance(wl, ref["flux"], wl.n_samples, False)
    err = np.abs(got["flux"] - ref["flux"])
    assert np.all(err <= tol), f"flux: worst err/tol {np.max(err / tol):.3g}"
    tolc = sbgpu.chi2_tolerance(wl, ref["flux"], tol, wl.n_samples, False)
    assert np.all(np.abs(got["chi2"] - ref["chi2"]) <= tolc)
    if grad:
        tol_d = sbgpu.grad_tolerance(wl, ref, wl.theta, wl.n_samples, False)
        assert np.all(np.abs(got["dflux"] - ref["dflux"]) <= tol_d), np.max(np.abs(got["dflux"] - ref["dflux"]) / tol_d, axis=0)
        told = sbgpu.dchi2_tolerance(wl, ref, tol, tol_d, wl.n_samples, False)
        assert np.all(np.abs(got["dchi2"] - ref["dchi2"]) <= told)


@pytest.mark.parametrize("config,n_sn", [(5, 400), (4, 300), (2, 500)])
def test_jittered_band_grids_run_the_node_weight_kernel(cuda_device, config, n_sn):
    wl = _prepare(workloads.make_workload(config, n_sn=n_sn, band_jitter=0.3))
    assert np.ptp(np.diff(wl.bands["wave"][:100])) > 1.0  # the grid really is non-uniform
    handles = sbgpu.load_handles(wl)
    ref = oracle.run_workload(wl, want_flux=True, want_chi2=True, want_dflux=True, want_dchi2=True)
    for mode in ("chi2", "grad"):
        got = sbgpu.run_gpu(wl, mode=mode, handles=handles)
        assert got["form"] == "tiled", got["form"]  # the library's own choice, not the direct kernel
        _check(wl, got, ref, mode == "grad")
        packed = sbgpu.run_gpu(wl, mode=mode, handles=handles, use_pack=True)
        assert np.array_equal(packed["flux"], got["flux"]) and np.array_equal(packed["chi2"], got["chi2"])
    direct = sbgpu.run_gpu(wl, mode="chi2", handles=handles, form="direct")
    tol = sbgpu.flux_tolerance(wl, ref["flux"], wl.n_samples, False)
    assert np.all(np.abs(direct["flux"] - got["flux"]) <= 2 * tol)


def _piecewise_bands(config):
    """Band grids with 5, 10 and 25 A stretches (tabulated filters often mix steps): far from the mean-step grid."""
    base = workloads.make_bands(config)
    out = []
    for b in range(len(base["offset"]) - 1):
        w = base["wave"][base["offset"][b]:base["offset"][b + 1]]
        lo, hi = w[0], w[-1]
        a, c = lo + 0.3 * (hi - lo), lo + 0.7 * (hi - lo)
        grid = np.concatenate([np.arange(lo, a, 25.0), np.arange(a, c, 5.0), np.arange(c, hi, 10.0), [hi]])
        grid = np.unique(grid)
        centre, sigma = 0.5 * (lo + hi), (hi - lo) / 3.0 / workloads.generators.FWHM_TO_SIGMA
        out.append((grid, np.exp(-0.5 * ((grid - centre) / sigma) ** 2)))
    return workloads.generators.pack_bands(out)


@pytest.mark.parametrize("config", [2, 5])
def test_piecewise_step_grids(cuda_device, config):
    wl = workloads.make_workload(config, n_sn=160, ragged=True)
    wl.bands = _piecewise_bands(config)
    _prepare(wl)
    ref = oracle.run_workload(wl, want_flux=True, want_chi2=True, want_dflux=True, want_dchi2=True)
    got = sbgpu.run_gpu(wl, mode="grad")
    assert got["form"] == "tiled"
    _check(wl, got, ref, True)
    got = sbgpu.run_gpu(wl, mode="chi2", use_pack=True)
    _check(wl, got, ref, False)


def test_samples_axis_and_colour_degree_7_on_jittered_grids(cuda_device):
    """n_cl = 8 (the degree-7 instantiation) and several parameter samples per supernova."""
    wl = workloads.make_workload(3, n_samples=384, band_jitter=0.25)
    rng = np.random.default_rng(5)
    wl.model = dict(wl.model)
    wl.model["cl_coef"] = np.concatenate([wl.model["cl_coef"], 0.02 * rng.standard_normal(3)])
    _prepare(wl)
    ref = oracle.run_workload(wl, want_flux=True, want_chi2=True)
    got = sbgpu.run_gpu(wl, mode="chi2")
    assert got["form"] == "tiled"
    _check(wl, got, ref, False)
