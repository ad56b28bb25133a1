"""Plain fp64 L-BFGS, one lane at a time -- the oracle of the batched device-resident fit driver.

TEST INFRASTRUCTURE, NOT PRODUCT (same rule as oracle/__init__.py).  PAPER.md:17 names the workload
("fmin_bfgs.py ... optimisation via L-BFGS-B"); the paper gives no algorithmic detail, so the algorithm
is the textbook one (Nocedal & Wright, Numerical Optimization, Alg. 7.4 two-loop recursion and Alg. 3.1
backtracking), restated here step by step.  Everything below is what DESIGN.md reading G16 fixes:

  variables   u_k = theta_k / s_k, s = (x0_start, 1, 1, 1): the fit works in scaled variables so that
              x0 ~ 1e-5 and the O(1) parameters share one metric; gradient g_u = g_theta * s.
  one EVALUATION = f and g at one trial point.  The lane is a state machine driven by evaluations:
    first evaluation at the start point: d = -g, alpha = min(1, 1 / ||g||_2).
    every later evaluation is at the trial point u_t = P(u + alpha d) (P = projection on the box, identity
    if no bounds) and is ACCEPTED if f_t is finite and f_t <= f + c1 * g.(u_t - u)   (Armijo, c1 = 1e-4):
      accepted   s = u_t - u, y = g_t - g; the pair is stored (circular memory m) if s.y > 1e-10 |s| |y|;
                 converged if f - f_t <= ftol * max(|f|, |f_t|, 1) or max_k |g_t,k| <= gtol;
                 d = -H g_t by the two-loop recursion with H0 = (s.y / y.y) I of the newest pair
                 (d = -g_t and alpha = min(1, 1/||g_t||) when the memory is empty or g_t.d >= 0: reset);
                 alpha = 1.
      rejected   alpha = alpha / 2; after 30 consecutive rejections the lane stops ("stalled").
    the lane also stops after max_eval evaluations or max_iter accepted steps.
Lanes are independent: the batched CUDA driver (sb_fit_lbfgs) runs the same machine for every unit with one
batched evaluation per step, so its per-lane sequence of evaluations is exactly this one.
"""
from __future__ import annotations

from typing import Callable, Dict, List, Optional, Tuple

import numpy as np

C1 = 1e-4
MAX_BACKTRACK = 30
CURV_EPS = 1e-10

RUNNING, CONVERGED, STALLED, EXHAUSTED = 0, 1, 2, 3


def _dot(a, b) -> float:
    s = 0.0
    for k in range(len(a)):  # fixed order: the CUDA driver sums in the same order
        s += float(a[k]) * float(b[k])
    return s


def two_loop(g: np.ndarray, S: List[np.ndarray], Y: List[np.ndarray]) -> np.ndarray:
    """-H g for the stored pairs (oldest first); Nocedal & Wright Alg. 7.4."""
    q = g.astype(np.float64).copy()
    m = len(S)
    alpha = [0.0] * m
    rho = [1.0 / _dot(Y[i], S[i]) for i in range(m)]
    for i in range(m - 1, -1, -1):
        alpha[i] = rho[i] * _dot(S[i], q)
        q = q - alpha[i] * Y[i]
    gamma = _dot(S[-1], Y[-1]) / _dot(Y[-1], Y[-1])
    r = gamma * q
    for i in range(m):
        beta = rho[i] * _dot(Y[i], r)
        r = r + (alpha[i] - beta) * S[i]
    return -r


def minimise(fun: Callable[[np.ndarray], Tuple[float, np.ndarray]], u0, *, memory: int = 8, max_eval: int = 60,
             max_iter: int = 1000, ftol: float = 1e-12, gtol: float = 0.0, lo=None, hi=None) -> Dict[str, object]:
    """Run the lane state machine on fun(u) -> (f, g).  Returns u, f, status, n_iter, n_eval and the
    trajectory of accepted f values (trace[0] = f at the start point)."""
    n = len(u0)
    lo = None if lo is None else np.asarray(lo, dtype=np.float64)
    hi = None if hi is None else np.asarray(hi, dtype=np.float64)

    def project(v):
        if lo is not None:
            v = np.maximum(v, lo)
        if hi is not None:
            v = np.minimum(v, hi)
        return v

    u = project(np.asarray(u0, dtype=np.float64).copy())
    f, g = fun(u)
    g = np.asarray(g, dtype=np.float64)
    n_eval, n_iter, n_back = 1, 0, 0
    trace = [float(f)]
    S: List[np.ndarray] = []
    Y: List[np.ndarray] = []
    status = RUNNING
    if not np.isfinite(f):
        status = STALLED
    gn = np.sqrt(_dot(g, g))
    if status == RUNNING and (gn == 0.0 or np.max(np.abs(g)) <= gtol):
        status = CONVERGED
    d = -g
    alpha = min(1.0, 1.0 / gn) if gn > 0.0 else 1.0
    while status == RUNNING:
        if n_eval >= max_eval or n_iter >= max_iter:
            status = EXHAUSTED
            break
        ut = project(u + alpha * d)
        ft, gt = fun(ut)
        gt = np.asarray(gt, dtype=np.float64)
        n_eval += 1
        step = ut - u
        if np.isfinite(ft) and ft <= f + C1 * _dot(g, step):
            y = gt - g
            sy = _dot(step, y)
            if sy > CURV_EPS * np.sqrt(_dot(step, step)) * np.sqrt(_dot(y, y)):
                S.append(step.copy())
                Y.append(y.copy())
                if len(S) > memory:
                    S.pop(0)
                    Y.pop(0)
            done = (f - ft) <= ftol * max(abs(f), abs(ft), 1.0) or np.max(np.abs(gt)) <= gtol
            u, f, g = ut, float(ft), gt
            n_iter += 1
            n_back = 0
            trace.append(f)
            if done:
                status = CONVERGED
                break
            reset = len(S) == 0
            if not reset:
                d = two_loop(g, S, Y)
                if _dot(g, d) >= 0.0:
                    reset = True
            if reset:
                S, Y = [], []
                d = -g
                gn = np.sqrt(_dot(g, g))
                alpha = min(1.0, 1.0 / gn) if gn > 0.0 else 1.0
            else:
                alpha = 1.0
        else:
            alpha *= 0.5
            n_back += 1
            if n_back >= MAX_BACKTRACK:
                status = STALLED
    return {"u": u, "f": f, "g": g, "status": status, "n_iter": n_iter, "n_eval": n_eval, "trace": np.array(trace)}


def fit_workload(wl, units=None, *, theta0=None, round_theta_to=None, **opts) -> Dict[str, np.ndarray]:
    """Fit (x0, x1, c, t0) of the given units (default: all; one parameter sample per supernova) of a
    workloads.Workload by minimising chi^2 (sbo_run with its analytic gradient) from theta0 (default
    wl.theta), one lane at a time.  round_theta_to = np.float32 rounds every trial theta to fp32 before the
    evaluation, as the CUDA driver does when the batch is fp32 (its kernels take fp32 parameters).
    Returns theta [n, 4], chi2 [n], status, n_iter, n_eval [n] and the list of chi^2 traces."""
    import oracle  # the C oracle's binding (this module lives beside it)

    th0 = wl.theta if theta0 is None else theta0
    assert wl.n_samples == 1 and len(th0["x0"]) == wl.n_sn
    units = np.arange(wl.n_sn) if units is None else np.asarray(units)
    model, bands = oracle.Model.from_dict(wl.model), oracle.Bands.from_dict(wl.bands)
    out = {"theta": np.zeros((len(units), 4)), "chi2": np.zeros(len(units)), "status": np.zeros(len(units), int),
           "n_iter": np.zeros(len(units), int), "n_eval": np.zeros(len(units), int), "trace": []}
    for k, s in enumerate(units):
        a, b = int(wl.obs_offset[s]), int(wl.obs_offset[s + 1])
        start = np.array([th0["x0"][s], th0["x1"][s], th0["c"][s], th0["t0"][s]], dtype=np.float64)
        scale = np.array([start[0], 1.0, 1.0, 1.0])

        def fun(u):
            th = u * scale
            if round_theta_to is not None:
                th = th.astype(round_theta_to).astype(np.float64)
            r = oracle.run(model, bands, n_sn=1, n_samples=1, obs_offset=[0, b - a], time=wl.time[a:b], band=wl.band[a:b],
                           zp=wl.zp[a:b], z=wl.z[s:s + 1], x0=th[0:1], x1=th[1:2], c=th[2:3], t0=th[3:4],
                           flux=wl.flux[a:b], fluxerr=wl.fluxerr[a:b], want_flux=False, want_chi2=True, want_dchi2=True,
                           threads=1)
            return float(r["chi2"][0]), r["dchi2"][0] * scale

        res = minimise(fun, start / scale, **opts)
        th = res["u"] * scale
        if round_theta_to is not None:
            th = th.astype(round_theta_to).astype(np.float64)
        out["theta"][k] = th
        out["chi2"][k] = res["f"]
        out["status"][k], out["n_iter"][k], out["n_eval"][k] = res["status"], res["n_iter"], res["n_eval"]
        out["trace"].append(res["trace"])
    return out
