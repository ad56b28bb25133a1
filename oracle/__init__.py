"""ctypes binding of the fp64 CPU oracle (oracle/salt_oracle.c).

TEST INFRASTRUCTURE, NOT PRODUCT: only tests/, __graft_entry__.smoke() and bench.py's
cpu_baseline / --impl reference legs import this.  It never imports the CUDA package and
the CUDA package never imports it.  Argument marshalling only; all arithmetic is in C.
"""
from __future__ import annotations

import ctypes as C
import os
import subprocess
from typing import Dict, Optional

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "salt_oracle.c")
_LIB = os.path.join(_HERE, "libsalt_oracle.so")

_dp = C.POINTER(C.c_double)
_ip = C.POINTER(C.c_int32)
_lp = C.POINTER(C.c_int64)


class _Model(C.Structure):
    _fields_ = [("n_phase", C.c_int32), ("n_wave", C.c_int32), ("phase", _dp), ("wave", _dp),
                ("m0", _dp), ("m1", _dp), ("n_cl", C.c_int32), ("cl_coef", _dp),
                ("cl_wave_b", C.c_double), ("cl_wave_v", C.c_double), ("cl_lo", C.c_double),
                ("cl_hi", C.c_double)]


class _Bands(C.Structure):
    _fields_ = [("n_bands", C.c_int32), ("offset", _lp), ("wave", _dp), ("trans", _dp)]


class _Batch(C.Structure):
    _fields_ = [("n_sn", C.c_int32), ("n_samples", C.c_int32), ("obs_offset", _ip), ("time", _dp),
                ("band", _ip), ("zp", _dp), ("z", _dp), ("x0", _dp), ("x1", _dp), ("c", _dp),
                ("t0", _dp)]


def build(force: bool = False) -> str:
    """Compile the oracle with gcc -O2 -fopenmp (as it stands; never tuned)."""
    if force or not os.path.exists(_LIB) or os.path.getmtime(_LIB) < os.path.getmtime(_SRC):
        cmd = ["gcc", "-O2", "-std=c99", "-fopenmp", "-fPIC", "-shared", "-o", _LIB, _SRC, "-lm"]
        subprocess.run(cmd, check=True)
    return _LIB


_lib = None


def lib():
    global _lib
    if _lib is None:
        L = C.CDLL(build())
        L.sbo_interp1.restype = C.c_double
        L.sbo_interp1.argtypes = [_dp, C.c_int64, C.c_int32, C.c_double, C.c_double, C.c_double, _dp]
        L.sbo_surface.restype = C.c_double
        L.sbo_surface.argtypes = [C.POINTER(_Model), C.c_int32, C.c_double, C.c_double, _dp]
        L.sbo_colour_law.restype = C.c_double
        L.sbo_colour_law.argtypes = [C.POINTER(_Model), C.c_double]
        L.sbo_trapz.restype = C.c_double
        L.sbo_trapz.argtypes = [_dp, _dp, C.c_int64]
        L.sbo_zpab.restype = C.c_double
        L.sbo_zpab.argtypes = [C.POINTER(_Bands), C.c_int32]
        L.sbo_eval.restype = C.c_double
        L.sbo_eval.argtypes = [C.POINTER(_Model), C.POINTER(_Bands), C.c_double, C.c_double,
                               C.c_int32, C.c_int32, C.c_double, C.c_double, C.c_double,
                               C.c_double, C.c_double, _dp]
        L.sbo_run.restype = C.c_int
        L.sbo_run.argtypes = [C.POINTER(_Model), C.POINTER(_Bands), C.POINTER(_Batch), _dp, _dp,
                              _dp, _dp, _dp, _dp]
        L.sbo_num_threads.restype = C.c_int
        L.sbo_set_num_threads.argtypes = [C.c_int]
        L.sbo_const_hc.restype = C.c_double
        _lib = L
    return _lib


def _f64(a) -> np.ndarray:
    return np.ascontiguousarray(np.asarray(a, dtype=np.float64))


def _ptr(a: Optional[np.ndarray], typ=_dp):
    return a.ctypes.data_as(typ) if a is not None else typ()


class Model:
    """Host-side model tables (fp64).  Keys as produced by workloads.make_model / make_colour_law."""

    def __init__(self, phase, wave, m0, m1, cl_coef, cl_wave_b, cl_wave_v, cl_lo, cl_hi):
        self.phase, self.wave = _f64(phase), _f64(wave)
        self.m0, self.m1 = _f64(m0), _f64(m1)
        assert self.m0.shape == (len(self.phase), len(self.wave)) == self.m1.shape
        self.cl_coef = _f64(cl_coef)
        self.c = _Model(len(self.phase), len(self.wave), _ptr(self.phase), _ptr(self.wave),
                        _ptr(self.m0), _ptr(self.m1), len(self.cl_coef), _ptr(self.cl_coef),
                        float(cl_wave_b), float(cl_wave_v), float(cl_lo), float(cl_hi))

    @classmethod
    def from_dict(cls, d: Dict[str, object]) -> "Model":
        return cls(d["phase"], d["wave"], d["m0"], d["m1"], d["cl_coef"], d["cl_wave_b"],
                   d["cl_wave_v"], d["cl_lo"], d["cl_hi"])

    def surface(self, which: int, p: float, lam_rest: float):
        d = C.c_double(0.0)
        v = lib().sbo_surface(C.byref(self.c), which, p, lam_rest, C.byref(d))
        return v, d.value

    def colour_law(self, lam_rest: float) -> float:
        return lib().sbo_colour_law(C.byref(self.c), lam_rest)


class Bands:
    def __init__(self, offset, wave, trans):
        self.offset = np.ascontiguousarray(np.asarray(offset, dtype=np.int64))
        self.wave, self.trans = _f64(wave), _f64(trans)
        self.c = _Bands(len(self.offset) - 1, _ptr(self.offset, _lp), _ptr(self.wave), _ptr(self.trans))

    @classmethod
    def from_dict(cls, d) -> "Bands":
        return cls(d["offset"], d["wave"], d["trans"])

    def zpab(self, b: int) -> float:
        return lib().sbo_zpab(C.byref(self.c), b)


def interp1(g, x0: float, dx: float, x: float):
    g = _f64(g)
    d = C.c_double(0.0)
    v = lib().sbo_interp1(_ptr(g), 1, len(g), x0, dx, x, C.byref(d))
    return v, d.value


def trapz(g, x) -> float:
    g, x = _f64(g), _f64(x)
    assert len(g) == len(x)
    return lib().sbo_trapz(_ptr(g), _ptr(x), len(g))


def eval_one(model: Model, bands: Bands, z, t, b, zp, x0, x1, c, t0, grad: bool = False):
    """One (supernova, sample, observation) band flux; zp=None means no zero-point scaling."""
    dm = (C.c_double * 4)()
    v = lib().sbo_eval(C.byref(model.c), C.byref(bands.c), z, t, b, 0 if zp is None else 1,
                       0.0 if zp is None else zp, x0, x1, c, t0, dm if grad else None)
    return (v, np.array(dm[:])) if grad else v


def run(model: Model, bands: Bands, *, n_sn, n_samples, obs_offset, time, band, zp, z, x0, x1, c,
        t0, flux=None, fluxerr=None, want_flux=True, want_dflux=False, want_chi2=False,
        want_dchi2=False, threads: Optional[int] = None) -> Dict[str, np.ndarray]:
    """Batched oracle; array layout identical to include/saltband.h (inputs up-cast to fp64)."""
    if threads:
        lib().sbo_set_num_threads(int(threads))
    obs_offset = np.ascontiguousarray(np.asarray(obs_offset, dtype=np.int32))
    band = np.ascontiguousarray(np.asarray(band, dtype=np.int32))
    time, z = _f64(time), _f64(z)
    zp = None if zp is None else _f64(zp)
    x0, x1, c, t0 = _f64(x0), _f64(x1), _f64(c), _f64(t0)
    n_tot = int(obs_offset[-1])
    n_units = n_sn * n_samples
    assert len(obs_offset) == n_sn + 1 and len(time) == n_tot == len(band) and len(z) == n_sn
    for a in (x0, x1, c, t0):
        assert len(a) == n_units
    flux = None if flux is None else _f64(flux)
    fluxerr = None if fluxerr is None else _f64(fluxerr)
    n_evals = n_tot * n_samples
    out = {}
    of = np.full(n_evals, np.nan) if want_flux else None
    od = np.full((n_evals, 4), np.nan) if want_dflux else None
    oc = np.full(n_units, np.nan) if want_chi2 else None
    og = np.full((n_units, 4), np.nan) if want_dchi2 else None
    bt = _Batch(n_sn, n_samples, _ptr(obs_offset, _ip), _ptr(time), _ptr(band, _ip), _ptr(zp),
                _ptr(z), _ptr(x0), _ptr(x1), _ptr(c), _ptr(t0))
    rc = lib().sbo_run(C.byref(model.c), C.byref(bands.c), C.byref(bt), _ptr(flux), _ptr(fluxerr),
                       _ptr(of), _ptr(od), _ptr(oc), _ptr(og))
    if rc != 0:
        raise ValueError("sbo_run: invalid arguments")
    if want_flux:
        out["flux"] = of
    if want_dflux:
        out["dflux"] = od
    if want_chi2:
        out["chi2"] = oc
    if want_dchi2:
        out["dchi2"] = og
    return out


def run_workload(wl, theta=None, **kw):
    """Convenience: run the oracle on a workloads.Workload (theta defaults to wl.theta)."""
    th = wl.theta if theta is None else theta
    n_samples = len(th["x0"]) // wl.n_sn
    return run(Model.from_dict(wl.model), Bands.from_dict(wl.bands), n_sn=wl.n_sn,
               n_samples=n_samples, obs_offset=wl.obs_offset, time=wl.time, band=wl.band,
               zp=wl.zp, z=wl.z, x0=th["x0"], x1=th["x1"], c=th["c"], t0=th["t0"],
               flux=wl.flux, fluxerr=wl.fluxerr, **kw)


def num_threads() -> int:
    return lib().sbo_num_threads()
