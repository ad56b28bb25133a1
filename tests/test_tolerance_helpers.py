"""-m "not gpu": the tolerance helper of the gradient tests (tests/sbgpu.py grad_term_sums) against the
oracle.  The helper measures the sum of ABSOLUTE terms of each derivative integral (reading G13a);
it interpolates the surfaces itself (vectorised), so it is pinned here: with the absolute values taken
away, the same code must reproduce the oracle's own dm/d(x1, c, t0) -- and its weights must equal
oracle.Model.surface point by point, border cells and out-of-grid points included."""
import numpy as np

import oracle
import sbgpu
import workloads


def test_stencil_equals_oracle_surface_pointwise():
    wl = workloads.make_workload(1)
    md = wl.model
    om = oracle.Model.from_dict(md)
    phase, wave = md["phase"], md["wave"]
    dp, dw = phase[1] - phase[0], wave[1] - wave[0]
    rng = np.random.default_rng(5)
    ps = np.concatenate([rng.uniform(phase[0] - 2, phase[-1] + 2, 60), [phase[0], phase[-1], phase[0] + 0.5 * dp, phase[-1] - 0.25 * dp, phase[3]]])
    ls = np.concatenate([rng.uniform(wave[0] - 50, wave[-1] + 50, 60), [wave[0], wave[-1], wave[0] + 0.3 * dw, wave[-1] - 0.6 * dw, wave[7]]])
    Wp, dWp = sbgpu._stencil((ps - phase[0]) / dp, len(phase))
    Wl, _ = sbgpu._stencil((ls - wave[0]) / dw, len(wave))
    for which, m in ((0, md["m0"]), (1, md["m1"])):
        val = np.einsum("ip,pw,iw->i", Wp, m, Wl)
        der = np.einsum("ip,pw,iw->i", dWp, m, Wl) / dp
        for i in range(len(ps)):
            v, d = om.surface(which, float(ps[i]), float(ls[i]))
            scale = np.abs(m).max()
            assert abs(val[i] - v) <= 1e-13 * scale and abs(der[i] - d) <= 1e-12 * scale / dp, (which, ps[i], ls[i])


def test_term_sums_without_the_absolute_value_are_the_oracle_gradient(monkeypatch):
    wl = workloads.make_workload(4, n_sn=6)
    ref = oracle.run_workload(wl, want_flux=True, want_dflux=True)
    A = sbgpu.grad_term_sums(wl, wl.theta, wl.n_samples)
    # bounds that any sum of absolute terms obeys
    assert np.all(A[:, 0] == 0.0) and np.all(A[:, 1:] >= np.abs(ref["dflux"][:, 1:]) * (1 - 1e-12))
    # signed: |.| replaced by the identity must give the derivative itself (x0 > 0 here)
    monkeypatch.setattr(sbgpu.np, "abs", lambda x: x)
    signed = sbgpu.grad_term_sums(wl, wl.theta, wl.n_samples)
    monkeypatch.undo()
    d = ref["dflux"]
    for q, sign in ((1, 1.0), (2, 1.0), (3, -1.0)):
        assert np.allclose(sign * signed[:, q], d[:, q], rtol=1e-10, atol=1e-12 * np.abs(d[:, q]).max()), q
