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


def _stencil(u_all: np.ndarray, n: int):
    """Dense interpolation weights of reading G1-G3 for grid coordinates u (in units of the grid step):
    Keys a = -1/2 in interior cells, linear in the first and last cell, zero outside [0, n-1].  Returns
    (W, dW), each [len(u), n]: value and d/du weights.  Tolerance helper only (checked against
    oracle.Model.surface by tests/test_tolerance_helpers.py); no expected value comes from here."""
    u_all = np.asarray(u_all, dtype=np.float64)
    W = np.zeros((len(u_all), n))
    dW = np.zeros_like(W)
    ok = (u_all >= 0.0) & (u_all <= n - 1)
    idx = np.nonzero(ok)[0]
    u = u_all[idx]
    i = np.minimum(np.floor(u).astype(np.int64), n - 2)
    t = u - i
    border = (i == 0) | (i == n - 2)
    kb, ki = idx[border], idx[~border]
    W[kb, i[border]] = 1.0 - t[border]
    W[kb, i[border] + 1] = t[border]
    dW[kb, i[border]] = -1.0
    dW[kb, i[border] + 1] = 1.0
    ti, ii = t[~border], i[~border]
    t2, t3 = ti * ti, ti * ti * ti
    for off, w, d in ((-1, (-t3 + 2 * t2 - ti) / 2, (-3 * t2 + 4 * ti - 1) / 2), (0, (3 * t3 - 5 * t2 + 2) / 2, (9 * t2 - 10 * ti) / 2),
                      (1, (-3 * t3 + 4 * t2 + ti) / 2, (-9 * t2 + 8 * ti + 1) / 2), (2, (t3 - t2) / 2, (3 * t2 - 2 * ti) / 2)):
        W[ki, ii + off] = w
        dW[ki, ii + off] = d
    return W, dW


def grad_term_sums(wl, th: Dict[str, np.ndarray], n_samples: int, use_zp: bool = True, row_terms: bool = True) -> np.ndarray:
    """[n_evals][4]: the sum of ABSOLUTE terms of each derivative's band integral (0 for x0), in out_flux order.
    With g_r[j] = the wavelength-interpolated model row r at band sample j, W_r / dW_r the phase weights and
    their derivatives, E = exp(c CL), k = T lam/(hc), w_j the trapezoid weights, S the zero-point factor:
        A_x1 = S x0 sum_j sum_r w_j |W_r M1_r[j]| E k,   A_c = S x0 sum_j sum_r w_j |W_r (M0 + x1 M1)_r[j] CL_j| E k,
        A_t0 = S x0/((1+z) dP) sum_j sum_r w_j |dW_r (M0 + x1 M1)_r[j]| E k
    (a derivative whose terms change sign is held to its sum of absolute term sizes, never to a
    cancelling total).  The phase rows are terms of their own: sum_r dW_r = 0, so dM/dp is a difference of
    neighbouring rows and cancels by construction, in ANY evaluation order.  row_terms=False takes the absolute
    value per sample after summing the rows (a smaller sum that ignores that cancellation; reported, not
    asserted).  The colour law and ZPAB come from the oracle's exposed pieces; the surfaces are interpolated
    here with _stencil."""
    import oracle

    md, bd = wl.model, wl.bands
    om, ob = oracle.Model.from_dict(md), oracle.Bands.from_dict(bd)
    phase, wave = np.asarray(md["phase"], dtype=np.float64), np.asarray(md["wave"], dtype=np.float64)
    m0, m1 = np.asarray(md["m0"], dtype=np.float64), np.asarray(md["m1"], dtype=np.float64)
    n_p, n_w = len(phase), len(wave)
    dp, dw = (phase[-1] - phase[0]) / (n_p - 1), (wave[-1] - wave[0]) / (n_w - 1)
    hc = 6.62607015e-27 * 2.99792458e18
    off = np.asarray(bd["offset"], dtype=np.int64)
    n_bands = len(off) - 1
    zpab = [ob.zpab(b) for b in range(n_bands)]
    out = np.zeros((int(wl.obs_offset[-1]) * n_samples, 4))
    for s in range(wl.n_sn):
        a, e = int(wl.obs_offset[s]), int(wl.obs_offset[s + 1])
        n_obs = e - a
        if n_obs == 0:
            continue
        opz = 1.0 + float(wl.z[s])
        bs = np.asarray(wl.band[a:e])
        tt = np.asarray(wl.time[a:e], dtype=np.float64)
        for b in np.unique(bs):
            if b < 0 or b >= n_bands:
                continue
            lam, tr = np.asarray(bd["wave"][off[b]:off[b + 1]], dtype=np.float64), np.asarray(bd["trans"][off[b]:off[b + 1]], dtype=np.float64)
            w = np.zeros_like(lam)
            w[:-1] += 0.5 * np.diff(lam)
            w[1:] += 0.5 * np.diff(lam)
            lr = lam / opz
            Wl, _ = _stencil((lr - wave[0]) / dw, n_w)            # [n_lam][n_wave]
            g0, g1 = m0 @ Wl.T, m1 @ Wl.T                          # [n_phase][n_lam]
            cl = np.array([om.colour_law(float(x)) for x in lr])
            wk = w * tr * lam / hc
            sel = np.nonzero(bs == b)[0]
            for k in range(n_samples):
                u = s * n_samples + k
                x0, x1, c, t0 = (float(th[q][u]) for q in ("x0", "x1", "c", "t0"))
                Wp, dWp = _stencil(((tt[sel] - t0) / opz - phase[0]) / dp, n_p)  # [n_sel][n_phase]
                ek = np.exp(c * cl) * wk
                sc = np.ones(len(sel))
                if use_zp:
                    sc = 10.0 ** (0.4 * np.asarray(wl.zp[a:e], dtype=np.float64)[sel]) / zpab[b]
                rows = a * n_samples + k * n_obs + sel
                g01 = g0 + x1 * g1
                if row_terms:  # |W_r| |g_r[j]|: absolute value of every (phase row, sample) term
                    out[rows, 1] = sc * abs(x0) * ((np.abs(Wp) @ np.abs(g1)) @ ek)
                    out[rows, 2] = sc * abs(x0) * (((np.abs(Wp) @ np.abs(g01)) * np.abs(cl)) @ ek)
                    out[rows, 3] = sc * abs(x0) / opz * (((np.abs(dWp) @ np.abs(g01)) / dp) @ ek)
                else:          # |sum_r W_r g_r[j]|: absolute value per sample, rows summed first
                    out[rows, 1] = sc * abs(x0) * (np.abs(Wp @ g1) @ ek)
                    out[rows, 2] = sc * abs(x0) * (np.abs((Wp @ g01) * cl) @ ek)
                    out[rows, 3] = sc * abs(x0) / opz * (np.abs((dWp @ g01) / dp) @ ek)
    return out


def grad_tolerance(wl, ref: Dict[str, np.ndarray], th: Dict[str, np.ndarray], n_samples: int, fp64: bool,
                   use_zp: bool = True):
    """Tolerance of d m/d(x0, x1, c, t0) (reading G13a): rel * (|dm| + A) + floor * peak/scale.

    The derivative integrands change sign inside the band (CL crosses zero at lambda_B, dM/dp at maximum
    light, M1 oscillates), so the integral can cancel far below the sum of its absolute terms, and rounding
    error scales with that sum, not with the total.  A is that sum, MEASURED per evaluation by
    grad_term_sums (0 for x0, whose integrand is the flux integrand itself)."""
    rel, floor = (1e-12, 1e-15) if fp64 else (1e-5, 1e-9)
    peak = unit_peaks(wl, ref["flux"], n_samples)
    scale = _theta_scale(wl, th, n_samples, len(ref["flux"]))
    A = grad_term_sums(wl, th, n_samples, use_zp)
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


def grad_conditioning(wl, ref: Dict[str, np.ndarray], th: Dict[str, np.ndarray], n_samples: int) -> np.ndarray:
    """|dm/dtheta| / A per evaluation and component (A = grad_term_sums, the sum of absolute terms of the
    derivative integral; inf for x0, whose integrand is the flux integrand itself): 1 means no cancellation,
    small values mean the integral cancels and no tolerance relative to the total can hold in fp32
    (reading G13a)."""
    A = grad_term_sums(wl, th, n_samples)
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
