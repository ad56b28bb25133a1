"""Seeded synthetic workloads for the five BASELINE.json configs.

Everything here is either a random draw (numpy ``default_rng(seed)``, PCG64) or a
closed-form table (Gaussian filters, a Planck-shaped surface).  None of the
method's arithmetic (rest-frame shift, interpolation, colour law, band integral,
zero point, chi^2) lives here, so both the CUDA path and the oracle may import it.

Recipe source: BASELINE.json `configs` (shapes, ranges, distributions) and
SURVEY.md section 8(d) (the choices BASELINE.json leaves open: surface formula,
colour-law draw, filter half-width, seeds).  Restated in DESIGN.md "Input recipe".

The paper runs on trained SALT3 / SALT3-NIR surfaces, survey filters
and real light curves; none of them are in this container, so these synthetic
inputs of the same shapes (71 x 901 / 71 x 1801 grids at 1 d x 10 A, 5 A filter
sampling, tens of epochs in 4-10 filters) stand in for them.
"""
from __future__ import annotations

from dataclasses import dataclass, field
from typing import Dict, Optional

import numpy as np

CONFIG_IDS = (1, 2, 3, 4, 5)

SEED_MODEL = 1001
SEED_COLOUR = 1002
SEED_CONFIG = {1: 2001, 2: 2002, 3: 2003, 4: 2004, 5: 2005}

# Colour-law reference wavelengths (B and V effective wavelengths, Angstrom) and the
# polynomial's validity range (BASELINE.json configs[0]: "linear extrapolation outside
# 2800-7000 A").
CL_WAVE_B = 4302.57
CL_WAVE_V = 5428.55
CL_LO = 2800.0
CL_HI = 7000.0

FWHM_TO_SIGMA = 2.3548200450309493  # 2*sqrt(2 ln 2)


def _smoothstep(x: np.ndarray) -> np.ndarray:
    x = np.clip(x, 0.0, 1.0)
    return x * x * (3.0 - 2.0 * x)


def make_model(nir: bool = False, seed: int = SEED_MODEL) -> Dict[str, np.ndarray]:
    """Synthetic SALT3-shaped M0/M1 node tables (fp64).

    Grid: phase -20..+50 d at 1 d (71 nodes); wavelength 2000..11000 A at 10 A
    (901 nodes), or 2000..20000 A (1801 nodes) for the SALT3-NIR-like config 5.
    M0: Gaussian-in-phase x Planck-shaped-in-wavelength, tapered to exactly zero at
    both wavelength edges.  M1: a seeded smooth cosine field at 0.1x the scale of M0.
    """
    rng = np.random.default_rng(seed)
    phase = -20.0 + np.arange(71, dtype=np.float64)
    n_wave = 1801 if nir else 901
    wave = 2000.0 + 10.0 * np.arange(n_wave, dtype=np.float64)
    p = phase[:, None]
    lam = wave[None, :]
    s = np.where(p < 0.0, 8.0, 16.0)
    g = np.exp(-0.5 * (p / s) ** 2)
    planck = lam ** -5.0 / np.expm1(1.438777e8 / (lam * 1.0e4))
    planck = planck / planck.max()
    taper = _smoothstep((lam - wave[0]) / 500.0) * _smoothstep((wave[-1] - lam) / 500.0)
    m0 = g * planck * taper
    a = rng.standard_normal(8) / np.sqrt(8.0)
    u = rng.integers(0, 4, size=8)
    v = rng.integers(0, 4, size=8)
    phi = rng.uniform(0.0, 2.0 * np.pi, size=8)
    fld = np.zeros_like(m0)
    for k in range(8):
        fld += a[k] * np.cos(
            2.0 * np.pi * (u[k] * (p + 20.0) / 70.0 + v[k] * (lam - wave[0]) / (wave[-1] - wave[0]))
            + phi[k]
        )
    m1 = 0.1 * m0 * fld
    return {
        "phase": np.ascontiguousarray(phase),
        "wave": np.ascontiguousarray(wave),
        "m0": np.ascontiguousarray(m0),
        "m1": np.ascontiguousarray(m1),
    }


def make_colour_law(seed: int = SEED_COLOUR) -> Dict[str, object]:
    """Seeded degree-4 colour-law polynomial in reduced wavelength l=(lam-B)/(V-B).

    a0 = 0, a1 = 1 - a2 - a3 - a4 (so the polynomial is 1 at l = 1), all scaled by
    0.4 ln 10 so the colour parameter is a magnitude.  Redrawn while the slope at
    either end of the 2800-7000 A range exceeds 1.5 (before scaling).
    """
    rng = np.random.default_rng(seed)
    l_lo = (CL_LO - CL_WAVE_B) / (CL_WAVE_V - CL_WAVE_B)
    l_hi = (CL_HI - CL_WAVE_B) / (CL_WAVE_V - CL_WAVE_B)
    while True:
        a2 = rng.uniform(-0.3, 0.0)
        a3 = rng.uniform(0.0, 0.1)
        a4 = rng.uniform(-0.015, 0.0)
        a1 = 1.0 - a2 - a3 - a4
        coef = np.array([0.0, a1, a2, a3, a4])

        def slope(x):
            return a1 + 2 * a2 * x + 3 * a3 * x * x + 4 * a4 * x ** 3

        if abs(slope(l_lo)) <= 1.5 and abs(slope(l_hi)) <= 1.5:
            break
    coef = coef * 0.9210340371976184  # 0.4 ln 10
    return {
        "cl_coef": coef,
        "cl_wave_b": CL_WAVE_B,
        "cl_wave_v": CL_WAVE_V,
        "cl_lo": CL_LO,
        "cl_hi": CL_HI,
    }


def gaussian_band(centre: float, fwhm: float, step: float = 5.0):
    """Gaussian transmission sampled at `step` A on centre +- H, H = step*round(1.5 FWHM/step)."""
    n_half = int(round(1.5 * fwhm / step))
    k = np.arange(-n_half, n_half + 1, dtype=np.float64)
    wave = centre + step * k
    sigma = fwhm / FWHM_TO_SIGMA
    trans = np.exp(-0.5 * ((wave - centre) / sigma) ** 2)
    return wave, trans


def pack_bands(bands) -> Dict[str, np.ndarray]:
    """CSR-pack a list of (wave, trans) pairs: band b owns [offset[b], offset[b+1])."""
    offset = np.zeros(len(bands) + 1, dtype=np.int64)
    for b, (w, _) in enumerate(bands):
        offset[b + 1] = offset[b] + len(w)
    wave = np.concatenate([np.asarray(w, dtype=np.float64) for w, _ in bands])
    trans = np.concatenate([np.asarray(t, dtype=np.float64) for _, t in bands])
    return {"offset": offset, "wave": np.ascontiguousarray(wave), "trans": np.ascontiguousarray(trans)}


def jitter_band_grids(bands: Dict[str, np.ndarray], jitter: float, seed: int = 1003) -> Dict[str, np.ndarray]:
    """Non-uniformly sampled copies of the band tables: every interior grid point is moved by U(-jitter,
    +jitter) x the local step (jitter < 0.5 keeps the grid strictly increasing; the end points stay), and the
    Gaussian transmission is re-tabulated at the moved wavelengths.  Real filter tables are not
    uniformly sampled; this is their synthetic stand-in.  Table generation only."""
    if not 0.0 <= jitter < 0.5:
        raise ValueError("jitter must be in [0, 0.5)")
    rng = np.random.default_rng(seed)
    wave, trans = bands["wave"].copy(), bands["trans"].copy()
    off = bands["offset"]
    for b in range(len(off) - 1):
        lo, hi = int(off[b]), int(off[b + 1])
        w = wave[lo:hi]
        step = (w[-1] - w[0]) / (len(w) - 1)
        centre = 0.5 * (w[0] + w[-1])
        sigma = (w[-1] - w[0]) / 3.0 / FWHM_TO_SIGMA  # the grid spans centre +- 1.5 FWHM (gaussian_band)
        w[1:-1] += rng.uniform(-jitter, jitter, size=len(w) - 2) * step
        trans[lo:hi] = np.exp(-0.5 * ((w - centre) / sigma) ** 2)
    return {"offset": off.copy(), "wave": wave, "trans": trans}


def make_bands(config: int) -> Dict[str, np.ndarray]:
    if config in (1, 3):
        centres = np.array([4800.0, 6200.0, 7500.0, 8700.0])
        fwhm = np.full(4, 1000.0)
    elif config == 2:
        centres = np.linspace(3600.0, 9000.0, 6)
        fwhm = np.linspace(800.0, 1200.0, 6)
    elif config == 4:
        centres = np.linspace(3600.0, 9000.0, 8)
        fwhm = np.linspace(800.0, 1200.0, 8)
    elif config == 5:
        centres = np.linspace(3600.0, 16000.0, 10)
        fwhm = np.linspace(800.0, 1600.0, 10)
    else:
        raise ValueError(f"unknown config {config}")
    return pack_bands([gaussian_band(c, f) for c, f in zip(centres, fwhm)])


@dataclass
class Workload:
    """One BASELINE.json config, as flat arrays in the layout of `sb_batch` (include/saltband.h).

    Observation and parameter arrays are fp32-representable values: they are
    generated in fp64, rounded to fp32 once, and that exact value is what both the CUDA
    path (fp32 or fp64 mode) and the oracle (which up-casts) receive.
    """

    config: int
    name: str
    model: Dict[str, object]
    bands: Dict[str, np.ndarray]
    n_sn: int
    n_samples: int
    obs_offset: np.ndarray  # int32 [n_sn+1]
    time: np.ndarray  # f32 [n_obs_total]
    band: np.ndarray  # i32 [n_obs_total]
    zp: np.ndarray  # f32 [n_obs_total]
    z: np.ndarray  # f32 [n_sn]
    theta_true: Dict[str, np.ndarray]  # each f32 [n_sn]
    theta: Dict[str, np.ndarray]  # each f32 [n_sn*n_samples], sample fastest
    noise: np.ndarray  # f64 [n_obs_total], standard normal
    flux: Optional[np.ndarray] = None  # f32 [n_obs_total], set by attach_data
    fluxerr: Optional[np.ndarray] = None
    meta: Dict[str, object] = field(default_factory=dict)

    @property
    def n_obs_total(self) -> int:
        return int(self.obs_offset[-1])

    @property
    def n_evals(self) -> int:
        return self.n_obs_total * self.n_samples

    @property
    def n_bands(self) -> int:
        return len(self.bands["offset"]) - 1


def _f32(x) -> np.ndarray:
    return np.ascontiguousarray(np.asarray(x, dtype=np.float64).astype(np.float32))


_NAMES = {
    1: "config1_smallest",
    2: "config2_batched_fit",
    3: "config3_nested_sampling",
    4: "config4_forward_grad",
    5: "config5_survey_nir",
}

_FULL = {  # n_sn, n_samples, n_obs per SN
    1: (1, 1, 40),
    2: (1024, 1, 60),
    3: (1, 65536, 50),
    4: (4096, 1, 100),
    5: (100000, 1, 80),
}


def make_workload(config: int, n_sn: Optional[int] = None, n_samples: Optional[int] = None,
                  ragged: bool = False, seed_offset: int = 0, band_jitter: float = 0.0) -> Workload:
    """Build config `config` (1..5).  `n_sn` / `n_samples` shrink it for parity tests.

    The shrunk workload is a prefix of the same random streams only in distribution, not
    element-wise; parity tests always hand identical arrays to both sides, so that is fine.
    `ragged=True` draws a different observation count per supernova (between half and the
    full count) to exercise the CSR layout; BASELINE.json's configs are all regular.
    `seed_offset` shifts the config's seed (one shard per rank in multi-GPU weak scaling).
    `band_jitter` > 0 replaces the 5 A band grids by non-uniform ones (jitter_band_grids).
    """
    if config not in CONFIG_IDS:
        raise ValueError(f"unknown config {config}")
    full_sn, full_samples, n_obs = _FULL[config]
    n_sn = full_sn if n_sn is None else int(n_sn)
    n_samples = full_samples if n_samples is None else int(n_samples)
    rng = np.random.default_rng(SEED_CONFIG[config] + int(seed_offset))

    model = make_model(nir=(config == 5))
    model.update(make_colour_law())
    bands = make_bands(config)
    if band_jitter > 0.0:
        bands = jitter_band_grids(bands, band_jitter)
    n_bands = len(bands["offset"]) - 1

    if ragged:
        counts = rng.integers(n_obs // 2, n_obs + 1, size=n_sn)
    else:
        counts = np.full(n_sn, n_obs, dtype=np.int64)
    obs_offset = np.zeros(n_sn + 1, dtype=np.int64)
    obs_offset[1:] = np.cumsum(counts)
    n_tot = int(obs_offset[-1])
    if n_tot >= 2 ** 31:
        raise ValueError("observation count overflows int32 CSR offsets")

    time = rng.uniform(-15.0, 45.0, size=n_tot)
    # band index round-robin within each supernova (BASELINE.json configs[0])
    band = np.concatenate([np.arange(c) % n_bands for c in counts]).astype(np.int32) if n_tot else np.zeros(0, np.int32)
    zp = np.full(n_tot, 25.0)
    noise = rng.standard_normal(n_tot)

    if config == 1:
        z = np.full(n_sn, 0.05)
        tt = {"x0": np.full(n_sn, 1e-5), "x1": np.full(n_sn, 0.5), "c": np.full(n_sn, 0.05),
              "t0": np.full(n_sn, 0.0)}
    elif config == 3:
        z = np.full(n_sn, 0.3)
        tt = {"x0": np.full(n_sn, 1e-5), "x1": np.full(n_sn, 0.5), "c": np.full(n_sn, 0.05),
              "t0": np.full(n_sn, 0.0)}
    else:
        z_hi = {2: 0.8, 4: 1.0, 5: 1.2}[config]
        t0_hi = 3.0 if config == 4 else 5.0
        z = rng.uniform(0.01, z_hi, size=n_sn)
        tt = {
            "x0": 10.0 ** rng.uniform(-6.0, -4.0, size=n_sn),
            "x1": rng.standard_normal(n_sn),
            "c": 0.1 * rng.standard_normal(n_sn),
            "t0": rng.uniform(-t0_hi, t0_hi, size=n_sn),
        }

    if config == 3:
        n = n_sn * n_samples
        th = {
            "x0": 10.0 ** rng.uniform(-6.0, -4.0, size=n),
            "x1": rng.uniform(-3.0, 3.0, size=n),
            "c": rng.uniform(-0.3, 0.3, size=n),
            "t0": rng.uniform(-10.0, 10.0, size=n),
        }
    elif config == 4:
        # one L-BFGS-B iterate: a perturbed start, so gradients are away from their zero
        def rep(a):
            return np.repeat(a, n_samples)

        n = n_sn * n_samples
        th = {
            "x0": rep(tt["x0"]) * np.exp(0.1 * rng.standard_normal(n)),
            "x1": rep(tt["x1"]) + 0.3 * rng.standard_normal(n),
            "c": rep(tt["c"]) + 0.03 * rng.standard_normal(n),
            "t0": rep(tt["t0"]) + np.clip(0.5 * rng.standard_normal(n), -2.0, 2.0),
        }
    else:
        th = {k: np.repeat(v, n_samples) for k, v in tt.items()}

    return Workload(
        config=config,
        name=_NAMES[config],
        model=model,
        bands=bands,
        n_sn=n_sn,
        n_samples=n_samples,
        obs_offset=obs_offset.astype(np.int32),
        time=_f32(time),
        band=np.ascontiguousarray(band, dtype=np.int32),
        zp=_f32(zp),
        z=_f32(z),
        theta_true={k: _f32(v) for k, v in tt.items()},
        theta={k: _f32(v) for k, v in th.items()},
        noise=noise,
        meta={"n_obs_per_sn": n_obs, "ragged": ragged, "seed": SEED_CONFIG[config] + int(seed_offset)},
    )


def attach_data(wl: Workload, model_flux_true: np.ndarray) -> Workload:
    """Set the photometry: f = m_true + sigma * N(0,1), sigma = max(5% |m_true|, 1e-3 max|m_true|).

    `model_flux_true` is the model band flux at theta_true for every observation
    ([n_obs_total], one sample per supernova), computed by the CALLER: tests pass the
    oracle's value, bench.py's GPU leg passes the CUDA path's.  No model arithmetic here.
    The floor keeps sigma > 0 when a band falls outside the model grid (flux 0).
    """
    m = np.asarray(model_flux_true, dtype=np.float64)
    if m.shape != (wl.n_obs_total,):
        raise ValueError("model_flux_true must be [n_obs_total]")
    sigma = np.empty_like(m)
    for s in range(wl.n_sn):
        a, b = int(wl.obs_offset[s]), int(wl.obs_offset[s + 1])
        if b > a:
            peak = np.max(np.abs(m[a:b]))
            floor = 1e-3 * peak if peak > 0 else 1.0
            sigma[a:b] = np.maximum(0.05 * np.abs(m[a:b]), floor)
    wl.flux = _f32(m + sigma * wl.noise)
    wl.fluxerr = _f32(sigma)
    return wl


def subset(wl: Workload, sn_index) -> Workload:
    """The supernovae `sn_index` (any order) of `wl` as their own Workload: same tables, the
    selected observation and parameter slices copied in that order.  Index bookkeeping only."""
    idx = np.asarray(sn_index, dtype=np.int64)
    ns = wl.n_samples
    n_obs = np.diff(wl.obs_offset).astype(np.int64)
    off = np.zeros(len(idx) + 1, dtype=np.int64)
    off[1:] = np.cumsum(n_obs[idx])
    if len(idx):
        sel = np.concatenate([np.arange(wl.obs_offset[s], wl.obs_offset[s + 1], dtype=np.int64) for s in idx])
    else:
        sel = np.zeros(0, dtype=np.int64)
    usel = (idx[:, None] * ns + np.arange(ns, dtype=np.int64)[None, :]).ravel()
    sub = Workload(
        config=wl.config, name=f"{wl.name}[subset {len(idx)}]", model=wl.model, bands=wl.bands, n_sn=len(idx),
        n_samples=ns, obs_offset=off.astype(np.int32), time=wl.time[sel].copy(), band=wl.band[sel].copy(),
        zp=wl.zp[sel].copy(), z=wl.z[idx].copy(), theta_true={k: v[idx].copy() for k, v in wl.theta_true.items()},
        theta={k: v[usel].copy() for k, v in wl.theta.items()}, noise=wl.noise[sel].copy(), meta=dict(wl.meta))
    if wl.flux is not None:
        sub.flux, sub.fluxerr = wl.flux[sel].copy(), wl.fluxerr[sel].copy()
    return sub


def shard_bounds(n_sn: int, weight: np.ndarray, world: int):
    """Contiguous partition of supernovae 0..n_sn over `world` ranks balanced by `weight` (e.g. the
    observations per supernova): bounds[r] .. bounds[r+1] is rank r's range."""
    w = np.asarray(weight, dtype=np.float64)
    if w.shape != (n_sn,):
        raise ValueError("weight must be [n_sn]")
    cum = np.concatenate([[0.0], np.cumsum(w)])
    total = cum[-1]
    bounds = [0]
    for r in range(1, world):
        target = total * r / world
        bounds.append(int(np.clip(np.searchsorted(cum, target, side="left"), bounds[-1], n_sn)))
    bounds.append(n_sn)
    return bounds
