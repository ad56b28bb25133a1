"""Pins of the L-BFGS oracle (oracle/lbfgs.py), the reference of the device-resident fit driver
("optimisation via L-BFGS-B"; reading G16).  None of these compares the oracle with
itself: the expected values are closed-form minimisers, the textbook Rosenbrock minimum, and theta_true
of noise-free synthetic photometry."""
import numpy as np
import pytest

import oracle
import workloads
from oracle import lbfgs


def test_spd_quadratic_reaches_the_closed_form_minimiser():
    rng = np.random.default_rng(3)
    for n in (2, 4, 7):
        A = rng.normal(size=(n, n))
        H = A @ A.T + n * np.eye(n)
        b = rng.normal(size=n)
        x_star = np.linalg.solve(H, b)  # minimiser of 1/2 x'Hx - b'x

        def fun(x):
            return 0.5 * x @ H @ x - b @ x, H @ x - b

        res = lbfgs.minimise(fun, rng.normal(size=n), memory=8, max_eval=200, ftol=0.0, gtol=1e-10)
        assert res["status"] == lbfgs.CONVERGED
        assert np.allclose(res["u"], x_star, rtol=0, atol=1e-8 * max(1.0, np.abs(x_star).max()))
        assert np.all(np.diff(res["trace"]) <= 0.0)  # Armijo: monotone
        # exact line searches would need n steps; backtracking L-BFGS stays within a few times n
        assert res["n_iter"] <= 12 * n


def test_rosenbrock_minimum():
    def fun(x):
        f = 100.0 * (x[1] - x[0] ** 2) ** 2 + (1.0 - x[0]) ** 2
        g = np.array([-400.0 * x[0] * (x[1] - x[0] ** 2) - 2.0 * (1.0 - x[0]), 200.0 * (x[1] - x[0] ** 2)])
        return f, g

    res = lbfgs.minimise(fun, np.array([-1.2, 1.0]), max_eval=400, ftol=0.0, gtol=1e-9)
    assert res["status"] == lbfgs.CONVERGED
    assert np.allclose(res["u"], [1.0, 1.0], atol=1e-7) and res["f"] < 1e-14
    assert np.all(np.diff(res["trace"]) <= 0.0)


def test_box_projection_stops_at_the_bound():
    # minimum of (x - 3)^2 + (y + 2)^2 on the box [0, 1] x [0, 1] is the corner (1, 0)
    def fun(x):
        return (x[0] - 3.0) ** 2 + (x[1] + 2.0) ** 2, np.array([2.0 * (x[0] - 3.0), 2.0 * (x[1] + 2.0)])

    res = lbfgs.minimise(fun, np.array([0.5, 0.5]), lo=[0.0, 0.0], hi=[1.0, 1.0], max_eval=100, ftol=1e-15)
    assert np.allclose(res["u"], [1.0, 0.0], atol=1e-12) and abs(res["f"] - 8.0) < 1e-12


def test_memory_is_bounded_and_evaluation_budget_is_respected():
    calls = []

    def fun(x):
        calls.append(1)
        return float(np.sum(x ** 4 + x ** 2)), 4.0 * x ** 3 + 2.0 * x

    res = lbfgs.minimise(fun, np.full(6, 2.0), memory=3, max_eval=9, ftol=0.0)
    assert res["n_eval"] == 9 == len(calls) and res["status"] == lbfgs.EXHAUSTED


def test_recovers_theta_true_on_noise_free_salt_photometry():
    """Config-4 shape: noise-free data at theta_true, start at the perturbed theta of the workload."""
    wl = workloads.make_workload(4, n_sn=6)
    true = oracle.run_workload(wl, theta={k: v.copy() for k, v in wl.theta_true.items()})["flux"]
    wl.noise = np.zeros(wl.n_obs_total)
    workloads.attach_data(wl, true)
    res = lbfgs.fit_workload(wl, max_eval=200, ftol=1e-15)
    tt = np.stack([wl.theta_true[k].astype(np.float64) for k in ("x0", "x1", "c", "t0")], axis=1)
    scale = np.stack([np.abs(tt[:, 0]), np.ones(6), np.ones(6), np.ones(6)], axis=1)
    assert np.all(np.abs(res["theta"] - tt) <= 1e-5 * scale), np.max(np.abs(res["theta"] - tt) / scale, axis=0)
    start = oracle.run_workload(wl, want_flux=False, want_chi2=True)["chi2"]
    assert np.all(res["chi2"] <= 1e-8 * start)
    for tr in res["trace"]:
        assert np.all(np.diff(tr) <= 0.0)  # monotone chi^2


def _pairs(rng, n, m):
    """m curvature pairs of a random SPD quadratic (y = H s, so s.y > 0), oldest first."""
    A = rng.normal(size=(n, n))
    H = A @ A.T + n * np.eye(n)
    S = [rng.normal(size=n) for _ in range(m)]
    return S, [H @ s for s in S]


def test_two_loop_satisfies_the_secant_equation():
    """The inverse-Hessian approximation built from pairs (s_i, y_i) maps the NEWEST y to its s, whatever
    the memory length (Nocedal & Wright eq. 6.6/7.16: H_{k+1} y_k = s_k); two_loop returns -H g."""
    rng = np.random.default_rng(11)
    for n, m in ((2, 1), (4, 3), (4, 8), (7, 5)):
        S, Y = _pairs(rng, n, m)
        d = lbfgs.two_loop(Y[-1], S, Y)
        assert np.allclose(d, -S[-1], rtol=0, atol=1e-12 * np.abs(S[-1]).max())


def test_two_loop_equals_the_dense_bfgs_update():
    """two_loop against the definition it is a fast form of: H_0 = gamma I with gamma of the newest pair, then
    H <- (I - rho s y')H(I - rho y s') + rho s s' for every pair, oldest first (Nocedal & Wright eq. 7.16 and
    7.20).  A wrong index, sign or loop order in the recursion changes H g for a generic g."""
    rng = np.random.default_rng(12)
    for n, m in ((3, 1), (4, 4), (6, 8)):
        S, Y = _pairs(rng, n, m)
        gamma = (S[-1] @ Y[-1]) / (Y[-1] @ Y[-1])
        H = gamma * np.eye(n)
        for s, y in zip(S, Y):
            rho = 1.0 / (y @ s)
            V = np.eye(n) - rho * np.outer(y, s)
            H = V.T @ H @ V + rho * np.outer(s, s)
        for _ in range(3):
            g = rng.normal(size=n)
            want = -H @ g
            assert np.allclose(lbfgs.two_loop(g, S, Y), want, rtol=0, atol=1e-11 * np.abs(want).max())
