"""-m gpu: the analytic gradient against SURVEY.md G13 AS WRITTEN (1e-5 |dm/dtheta| + 1e-9 max|m| /
theta-scale; 3e-5 for t0), beside the condition-aware form of DESIGN.md reading G13a that the other
gradient tests use.  The strict form is asserted wherever it can hold: for d/dx0 on every evaluation,
for all four components in fp64 mode, and in fp32 for x1, c, t0 on the evaluations whose derivative
integral does not cancel (|dm/dtheta| >= A / 10, A = the measured sum of absolute terms of the derivative
integral, sbgpu.grad_term_sums).  The worst error / tolerance ratios of every (config shape, formulation,
precision, component) are printed (pytest -s shows them): DESIGN.md section 2 quotes them."""
import numpy as np
import pytest

import oracle
import sbgpu
import workloads

pytestmark = pytest.mark.gpu

SHAPES = [(3, {"n_samples": 96}), (4, {"n_sn": 160}), (5, {"n_sn": 120})]
WELL = 0.1  # |dm| / A above which the derivative integral counts as non-cancelling (condition number <= 10)


def _prepare(config, **kw):
    wl = workloads.make_workload(config, **kw)
    true = oracle.run_workload(wl, theta={k: v.copy() for k, v in wl.theta_true.items()})["flux"]
    workloads.attach_data(wl, true)
    return wl


@pytest.mark.parametrize("config,kw", SHAPES)
def test_gradient_against_strict_g13(cuda_device, config, kw):
    wl = _prepare(config, **kw)
    ns = wl.n_samples
    ref = oracle.run_workload(wl, want_flux=True, want_dflux=True)
    cond = sbgpu.grad_conditioning(wl, ref, wl.theta, ns)
    for fp64 in (False, True):
        strict = sbgpu.grad_tolerance_strict(wl, ref, wl.theta, ns, fp64)
        loose = sbgpu.grad_tolerance(wl, ref, wl.theta, ns, fp64)
        rel = 1e-12 if fp64 else 1e-5  # the same bound with per-sample absolute values only (rows summed first)
        per_sample = loose + rel * (sbgpu.grad_term_sums(wl, wl.theta, ns, row_terms=False) - sbgpu.grad_term_sums(wl, wl.theta, ns))
        for form in ("direct",) if fp64 else ("direct", "tiled"):
            got = sbgpu.run_gpu(wl, mode="grad", fp64=fp64, form=form, with_data=False)
            assert got["form"] == form
            err = np.abs(got["dflux"] - ref["dflux"])
            ratio_all = np.max(err / strict, axis=0)
            well = cond >= WELL
            ratio_well = np.array([np.max((err / strict)[well[:, q], q]) if well[:, q].any() else 0.0 for q in range(4)])
            ratio_loose = np.max(err / loose, axis=0)
            key = f"config{config}:{form}:{'fp64' if fp64 else 'fp32'}"
            print(key, "strict(all)", np.round(ratio_all, 3), "strict(well)", np.round(ratio_well, 3), "G13a",
                  np.round(ratio_loose, 4), "G13a-per-sample", np.round(np.max(err / per_sample, axis=0), 3),
                  "well fraction", np.round(well.mean(axis=0), 3))
            assert np.all(ratio_loose <= 1.0), (key, ratio_loose)
            assert ratio_all[0] <= 1.0, (key, "x0 strict", ratio_all[0])
            if fp64:
                assert np.all(ratio_all <= 1.0), (key, "fp64 strict", ratio_all)
            else:
                assert np.all(ratio_well <= 1.0), (key, "fp32 strict on the non-cancelling subset", ratio_well)
