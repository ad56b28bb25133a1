"""-m gpu: random batch shapes through the node-weight kernel and the direct kernel -- two exact
re-associations of the same finite sums, each within the flux tolerance of the oracle,
so their results must agree within twice that tolerance whatever the shape.  No oracle in the loop: the cases
are cheap, so the seeds below cover what the structured tests do not combine -- 1 to 6000 supernovae (around
the multiples of 32 and of 32 x n_SM that fill whole groups and waves), 1 to 12 bands of random centre, width
and step, uniform or jittered grids, both model grids, ragged / empty / single huge light curves, phases
outside the grid, several parameter samples, forward or gradient, with or without a pack."""
import numpy as np
import pytest

import sbgpu
from workloads.generators import Workload, gaussian_band, jitter_band_grids, make_colour_law, make_model, pack_bands

pytestmark = pytest.mark.gpu


def _f32(a):
    return np.asarray(a, np.float64).astype(np.float32)


def random_workload(rng):
    n_sn = int(rng.choice([1, 2, 5, 31, 32, 33, 147, 148, 149, 500, 1500, 4736, 4737, 6000]))
    n_bands = int(rng.integers(1, 13))
    nir = bool(rng.integers(0, 2))
    model = make_model(nir=nir)
    model.update(make_colour_law())
    centres = np.sort(rng.uniform(3200.0, 16000.0 if nir else 9500.0, n_bands))
    fwhm = rng.uniform(300.0, 1800.0, n_bands)
    step = float(rng.choice([5.0, 5.0, 10.0, 2.5]))
    bands = pack_bands([gaussian_band(c, f, step) for c, f in zip(centres, fwhm)])
    if rng.integers(0, 2):
        bands = jitter_band_grids(bands, float(rng.uniform(0.05, 0.45)), seed=int(rng.integers(1, 1000)))
    kind = int(rng.integers(0, 4))
    if kind == 0:
        counts = np.full(n_sn, int(rng.integers(1, 130)))
    elif kind == 1:
        counts = rng.integers(0, 200, n_sn)
    elif kind == 2:  # one light curve larger than a round of the kernel
        counts = rng.integers(0, 60, n_sn)
        counts[rng.integers(0, n_sn)] = int(rng.integers(1500, 7000))
    else:
        counts = rng.integers(0, 12, n_sn)
    n_samples = int(rng.choice([1, 1, 1, 2, 7])) if n_sn * counts.sum() < 3e5 else 1
    off = np.zeros(n_sn + 1, np.int64)
    off[1:] = np.cumsum(counts)
    n_tot, n_u = int(off[-1]), n_sn * n_samples
    th = {"x0": 10.0 ** rng.uniform(-6, -4, n_u), "x1": rng.standard_normal(n_u), "c": 0.1 * rng.standard_normal(n_u),
          "t0": rng.uniform(-5, 5, n_u)}
    wl = Workload(config=0, name="random", model=model, bands=bands, n_sn=n_sn, n_samples=n_samples,
                  obs_offset=off.astype(np.int32), time=_f32(rng.uniform(-25.0, 60.0, n_tot)),
                  band=rng.integers(0, n_bands, n_tot).astype(np.int32), zp=_f32(np.full(n_tot, 25.0)),
                  z=_f32(rng.uniform(0.0, float(rng.choice([0.1, 0.8, 1.5])), n_sn)),
                  theta_true={k: _f32(v[::n_samples]) for k, v in th.items()}, theta={k: _f32(v) for k, v in th.items()},
                  noise=rng.standard_normal(n_tot), meta={})
    wl.flux, wl.fluxerr = _f32(rng.standard_normal(n_tot) * 1e3), _f32(np.full(n_tot, 50.0))
    return wl


@pytest.mark.parametrize("seed", range(5000, 5040))
def test_node_weight_and_direct_kernels_agree(cuda_device, seed):
    rng = np.random.default_rng(seed)
    wl = random_workload(rng)
    grad, pack = bool(rng.integers(0, 2)), bool(rng.integers(0, 2))
    if wl.n_obs_total == 0:
        pytest.skip("empty batch")
    handles = sbgpu.load_handles(wl)
    mode = "grad" if grad else "chi2"
    a = sbgpu.run_gpu(wl, mode=mode, form="tiled", handles=handles, use_pack=pack)
    b = sbgpu.run_gpu(wl, mode=mode, form="direct", handles=handles)
    assert a["form"] == "tiled" and b["form"] == "direct"
    fa, fb = a["flux"], b["flux"]
    assert np.array_equal(np.isnan(fa), np.isnan(fb))
    fin = np.isfinite(fb)
    peak = sbgpu.unit_peaks(wl, np.where(fin, fb, 0.0), wl.n_samples)
    tol = 2.0 * (1e-5 * np.abs(fb) + 1e-9 * peak) + 1e-300
    assert np.all((np.abs(fa - fb) <= tol)[fin]), float(np.max((np.abs(fa - fb) / tol)[fin]))
    assert np.allclose(a["chi2"], b["chi2"], rtol=2e-3, atol=1e-3, equal_nan=True)
    if grad:  # G13a-shaped bound between the two kernels (relative to the non-cancelling magnitude)
        m = np.abs(np.where(fin, fb, 0.0))[:, None]
        scale = np.abs(b["dflux"]) + m * np.array([0.0, 1.0, 1.0, 1.0])[None, :]
        n_obs = np.diff(wl.obs_offset)  # out_dflux layout: [supernova][sample][observation]
        x0 = np.concatenate([np.repeat(row, n) for row, n in zip(wl.theta["x0"].reshape(wl.n_sn, -1), n_obs)])
        floor = 1e-9 * peak[:, None] / np.stack([np.abs(x0), np.ones_like(x0), np.ones_like(x0), np.ones_like(x0)], axis=1)
        ok = np.abs(a["dflux"] - b["dflux"]) <= 4e-5 * scale + 2.0 * floor
        assert np.all(ok[fin]), "gradient of the two kernels differs"
