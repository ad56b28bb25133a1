"""Test helpers: run a workloads.Workload through the C-ABI CUDA library, and the tolerance rules
of DESIGN.md (reading G13).  Imported by the -m gpu tests and by __graft_entry__.smoke()."""
from __future__ import annotations

from typing import Dict, Optional

import numpy as np


def load_handles(wl):
    import paper_2504_08081_b200 as sb

    md, bd = wl.model, wl.bands
    model = sb.sb_load_model(md["phase"], md["wave"], md["m0"], md["m1"], md["cl_coef"], md["cl_wave_b"],
                             md["cl_wave_v"], md["cl_lo"], md["cl_hi"])
    bands = sb.sb_load_bandpasses(bd["offset"], bd["wave"], bd["trans"])
    return model, bands


def run_gpu(wl, *, mode: str = "chi2", fp64: bool = False, theta: Optional[Dict[str, np.ndarray]] = None,
            use_zp: bool = True, handles=None, want_flux: bool = True, want_dflux: bool = True,
            with_data: bool = True, form: Optional[str] = None, use_pack: bool = False) -> Dict[str, np.ndarray]:
    """mode: 'flux' (sb_bandflux), 'chi2' (sb_chi2), 'grad' (sb_bandflux_grad).  form: None (library's
    choice), 'direct' or 'grouped' (include/saltband.h SB_FORM_*).  Returns host fp64 arrays."""
    import torch

    import paper_2504_08081_b200 as sb

    dev = torch.device("cuda:0")
    ft = torch.float64 if fp64 else torch.float32
    dt = sb.SB_F64 if fp64 else sb.SB_F32
    dt |= {None: 0, "direct": sb.SB_FORM_DIRECT, "grouped": sb.SB_FORM_GROUPED, "tiled": sb.SB_FORM_TILED}[form]
    model, bands = handles if handles is not None else load_handles(wl)
    th = wl.theta if theta is None else theta
    n_units = len(th["x0"])
    n_samples = n_units // max(wl.n_sn, 1) if wl.n_sn else 1
    n_tot = wl.n_obs_total

    def dev_f(a):
        return torch.as_tensor(np.asarray(a, dtype=np.float64), dtype=ft).to(dev).contiguous()

    common = dict(
        dtype=dt, n_sn=wl.n_sn, n_samples=n_samples, n_obs_total=n_tot,
        obs_offset=torch.as_tensor(np.asarray(wl.obs_offset, dtype=np.int32)).to(dev),
        time=dev_f(wl.time), band=torch.as_tensor(np.asarray(wl.band, dtype=np.int32)).to(dev),
        zp=dev_f(wl.zp) if use_zp else None, z=dev_f(wl.z), x0=dev_f(th["x0"]), x1=dev_f(th["x1"]),
        c=dev_f(th["c"]), t0=dev_f(th["t0"]))
    if use_pack:  # include/saltband.h: sb_pack_observations (fp32 only), built on the current stream
        common["pack"] = sb.sb_pack_observations(model, bands, dtype=sb.SB_F32, n_sn=wl.n_sn, z=common["z"])
    out: Dict[str, np.ndarray] = {}
    nan = float("nan")
    o_flux = torch.full((n_tot * n_samples,), nan, dtype=ft, device=dev) if want_flux else None
    if mode == "flux":
        sb.sb_bandflux(model, bands, out_flux=o_flux, **common)
    elif mode == "chi2":
        o_chi = torch.full((n_units,), nan, dtype=ft, device=dev)
        sb.sb_chi2(model, bands, flux=dev_f(wl.flux), fluxerr=dev_f(wl.fluxerr), out_chi2=o_chi, out_flux=o_flux,
                   **common)
        out["chi2"] = o_chi.double().cpu().numpy()
    elif mode == "grad":
        o_d = torch.full((n_tot * n_samples * 4,), nan, dtype=ft, device=dev) if want_dflux else None
        data = with_data and wl.flux is not None
        o_chi = torch.full((n_units,), nan, dtype=ft, device=dev) if data else None
        o_dchi = torch.full((n_units * 4,), nan, dtype=ft, device=dev) if data else None
        sb.sb_bandflux_grad(model, bands, flux=dev_f(wl.flux) if data else None,
                            fluxerr=dev_f(wl.fluxerr) if data else None, out_flux=o_flux, out_dflux=o_d,
                            out_chi2=o_chi, out_dchi2=o_dchi, **common)
        if o_d is not None:
            out["dflux"] = o_d.double().cpu().numpy().reshape(-1, 4)
        if data:
            out["chi2"] = o_chi.double().cpu().numpy()
            out["dchi2"] = o_dchi.double().cpu().numpy().reshape(-1, 4)
    else:
        raise ValueError(mode)
    torch.cuda.synchronize()
    out["launches"] = sb.last_launch_count()
    out["form"] = sb.last_form()
    if o_flux is not None:
        out["flux"] = o_flux.double().cpu().numpy()
    return out


# ------------------------------------------------------------------ tolerances (G13)
def unit_peaks(wl, flux_ref: np.ndarray, n_samples: int) -> np.ndarray:
    """max_i |m_i| per evaluation's unit, broadcast to every evaluation (layout of out_flux)."""
    peak = np.empty_like(flux_ref)
    for s in range(wl.n_sn):
        a, b = int(wl.obs_offset[s]) * n_samples, int(wl.obs_offset[s + 1]) * n_samples
        n_obs = int(wl.obs_offset[s + 1] - wl.obs_offset[s])
        if n_obs == 0:
            continue
        blk = np.abs(flux_ref[a:b]).reshape(n_samples, n_obs)
        peak[a:b] = np.repeat(blk.max(axis=1), n_obs)
    return peak


def flux_tolerance(wl, flux_ref: np.ndarray, n_samples: int, fp64: bool) -> np.ndarray:
    """fp32: 1e-5 |m| + 1e-9 peak (BASELINE.json north_star); fp64: 1e-12 |m| + 1e-15 peak."""
    peak = unit_peaks(wl, flux_ref, n_samples)
    if fp64:
        return 1e-12 * np.abs(flux_ref) + 1e-15 * peak
    return 1e-5 * np.abs(flux_ref) + 1e-9 * peak


def chi2_tolerance(wl, flux_ref: np.ndarray, tol_flux: np.ndarray, n_samples: int, fp64: bool) -> np.ndarray:
    """Bound implied by perturbing each m_i by its tolerance, plus the output's own rounding."""
    out = np.zeros(wl.n_sn * n_samples)
    for s in range(wl.n_sn):
        a, b = int(wl.obs_offset[s]), int(wl.obs_offset[s + 1])
        n_obs = b - a
        for k in range(n_samples):
            sl = slice(a * n_samples + k * n_obs, a * n_samples + (k + 1) * n_obs)
            r = (wl.flux[a:b].astype(np.float64) - flux_ref[sl]) / wl.fluxerr[a:b]
            t = tol_flux[sl] / wl.fluxerr[a:b]
            chi = np.sum(r * r)
            out[s * n_samples + k] = np.sum(2.0 * np.abs(r) * t + t * t) + (1e-13 if fp64 else 1e-6) * chi
    return out


def grad_tolerance(wl, ref: Dict[str, np.ndarray], th: Dict[str, np.ndarray], n_samples: int, fp64: bool):
    """Tolerance of d m/d(x0, x1, c, t0) (reading G13a): rel * (|dm| + A) + floor * peak/scale.

    The derivative integrands change sign inside the band (CL crosses zero at lambda_B, dM/dp at
    maximum light, M1 oscillates), so the integral can cancel far below the sum of its absolute
    terms, and rounding error scales with that sum, not with the total.  A is that non-cancelling
    magnitude: 0 for x0, |m| for x1 and c (|M1| <~ |M0|, |CL| = O(1)), |m|/(dP (1+z)) for t0."""
    rel, floor = (1e-12, 1e-15) if fp64 else (1e-5, 1e-9)
    peak = unit_peaks(wl, ref["flux"], n_samples)
    m = np.abs(ref["flux"])
    dp = float(wl.model["phase"][1] - wl.model["phase"][0])
    scale = np.empty((len(ref["flux"]), 4))
    opz = np.empty(len(ref["flux"]))
    for s in range(wl.n_sn):
        a, b = int(wl.obs_offset[s]), int(wl.obs_offset[s + 1])
        n_obs = b - a
        opz[a * n_samples:b * n_samples] = 1.0 + float(wl.z[s])
        for k in range(n_samples):
            u = s * n_samples + k
            sl = slice(a * n_samples + k * n_obs, a * n_samples + (k + 1) * n_obs)
            scale[sl, 0] = abs(th["x0"][u])
            scale[sl, 1] = max(abs(th["x1"][u]), 1.0)
            scale[sl, 2] = max(abs(th["c"][u]), 1.0)
            scale[sl, 3] = max(abs(th["t0"][u]), 1.0)
    A = np.stack([np.zeros_like(m), m, m, m / (dp * opz)], axis=1)
    return rel * (np.abs(ref["dflux"]) + A) + floor * peak[:, None] / scale


def grad_tolerance_strict(wl, ref: Dict[str, np.ndarray], th: Dict[str, np.ndarray], n_samples: int, fp64: bool):
    """SURVEY.md G13 as written: 1e-5 |dm/dtheta| + 1e-9 max|m| / theta-scale (3e-5 for t0); fp64: 1e-12 / 1e-15.
    Relative to the derivative itself, so it is only attainable where the derivative integral does not
    cancel (see grad_conditioning); asserted on that subset, and on every evaluation for x0 and in fp64."""
    rel = np.array([1e-12] * 4) if fp64 else np.array([1e-5, 1e-5, 1e-5, 3e-5])
    floor = 1e-15 if fp64 else 1e-9
    peak = unit_peaks(wl, ref["flux"], n_samples)
    scale = _theta_scale(wl, th, n_samples, len(ref["flux"]))
    return rel[None, :] * np.abs(ref["dflux"]) + floor * peak[:, None] / scale


def grad_conditioning(wl, ref: Dict[str, np.ndarray], n_samples: int) -> np.ndarray:
    """|dm/dtheta| / A per evaluation and component (A = the non-cancelling magnitude of grad_tolerance;
    inf for x0, whose integrand is the flux integrand itself): small values mean the derivative integral
    cancels and no tolerance relative to the total can hold in fp32 (reading G13a)."""
    m = np.abs(ref["flux"])
    dp = float(wl.model["phase"][1] - wl.model["phase"][0])
    opz = np.repeat(1.0 + wl.z.astype(np.float64), np.diff(wl.obs_offset) * n_samples)
    A = np.stack([np.zeros_like(m), m, m, m / (dp * opz)], axis=1)
    with np.errstate(divide="ignore", invalid="ignore"):
        return np.where(A > 0, np.abs(ref["dflux"]) / A, np.inf)


def _theta_scale(wl, th, n_samples, n_ev):
    scale = np.empty((n_ev, 4))
    for s in range(wl.n_sn):
        a, b = int(wl.obs_offset[s]), int(wl.obs_offset[s + 1])
        n_obs = b - a
        for k in range(n_samples):
            u = s * n_samples + k
            sl = slice(a * n_samples + k * n_obs, a * n_samples + (k + 1) * n_obs)
            scale[sl, 0] = abs(th["x0"][u])
            scale[sl, 1] = max(abs(th["x1"][u]), 1.0)
            scale[sl, 2] = max(abs(th["c"][u]), 1.0)
            scale[sl, 3] = max(abs(th["t0"][u]), 1.0)
    return scale


def dchi2_tolerance(wl, ref: Dict[str, np.ndarray], tol_flux, tol_dflux, n_samples: int, fp64: bool) -> np.ndarray:
    """Propagate flux and dflux tolerances through -2 sum (f-m)/sigma^2 dm (sum of absolute terms)."""
    out = np.zeros((wl.n_sn * n_samples, 4))
    for s in range(wl.n_sn):
        a, b = int(wl.obs_offset[s]), int(wl.obs_offset[s + 1])
        n_obs = b - a
        f, e = wl.flux[a:b].astype(np.float64), wl.fluxerr[a:b].astype(np.float64)
        for k in range(n_samples):
            sl = slice(a * n_samples + k * n_obs, a * n_samples + (k + 1) * n_obs)
            res = np.abs(f - ref["flux"][sl])[:, None]
            dm = np.abs(ref["dflux"][sl])
            term = 2.0 / (e * e)[:, None] * (tol_flux[sl][:, None] * dm + res * tol_dflux[sl] + tol_flux[sl][:, None] * tol_dflux[sl])
            mag = 2.0 / (e * e)[:, None] * res * dm
            out[s * n_samples + k] = term.sum(axis=0) + (1e-13 if fp64 else 1e-6) * mag.sum(axis=0)
    return out
