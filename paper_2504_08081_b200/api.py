"""ctypes binding of libsaltband.so -- same names and argument meaning as include/saltband.h.

Marshalling only.  Loaders take host arrays (numpy, fp64); compute calls take CUDA torch tensors
and enqueue on torch's current stream.  Nothing here computes any step of the method.
"""
from __future__ import annotations

import ctypes as C
import os
from typing import Optional

import numpy as np

SB_F32, SB_F64 = 0, 1
SB_FORM_DIRECT, SB_FORM_GROUPED, SB_FORM_TILED = 0x100, 0x200, 0x400  # optional formulation bits OR-ed into dtype
SB_NOALLOC_MAX_SN = 131072  # include/saltband.h: largest n_sn sb_chi2_noalloc accepts

_PKG = os.path.dirname(os.path.abspath(__file__))
# SALTBAND_LIB=checked loads the bounds-checked build of the same sources (build.py --checked)
_LIB_PATH = os.path.join(_PKG, "libsaltband_checked.so" if os.environ.get("SALTBAND_LIB") == "checked" else "libsaltband.so")


class SaltbandError(RuntimeError):
    pass


class _Batch(C.Structure):
    _fields_ = [
        ("dtype", C.c_int32), ("n_sn", C.c_int32), ("n_samples", C.c_int32), ("n_obs_total", C.c_int32),
        ("obs_offset", C.c_void_p), ("time", C.c_void_p), ("band", C.c_void_p), ("zp", C.c_void_p),
        ("z", C.c_void_p), ("x0", C.c_void_p), ("x1", C.c_void_p), ("c", C.c_void_p), ("t0", C.c_void_p),
        ("pack", C.c_void_p),
    ]


class _FitOpts(C.Structure):
    _fields_ = [("memory", C.c_int32), ("max_eval", C.c_int32), ("max_iter", C.c_int32), ("trace_len", C.c_int32),
                ("ftol", C.c_double), ("gtol", C.c_double), ("lo", C.POINTER(C.c_double)), ("hi", C.POINTER(C.c_double))]


class _FitResult(C.Structure):
    _fields_ = [("theta", C.c_void_p), ("chi2", C.c_void_p), ("status", C.c_void_p), ("n_iter", C.c_void_p),
                ("n_eval", C.c_void_p), ("trace", C.c_void_p)]


FIT_RUNNING, FIT_CONVERGED, FIT_STALLED, FIT_EXHAUSTED = 0, 1, 2, 3  # sb_fit_result.status

_lib = None


def lib_path() -> str:
    return _LIB_PATH


def _load():
    global _lib
    if _lib is not None:
        return _lib
    if not os.path.exists(_LIB_PATH):
        raise ImportError(
            f"{_LIB_PATH} is missing: build it with `python -m paper_2504_08081_b200.build` "
            "(there is no CPU fallback)")
    L = C.CDLL(_LIB_PATH)
    dp, vp = C.POINTER(C.c_double), C.c_void_p
    L.sb_load_model.restype = C.c_int
    L.sb_load_model.argtypes = [dp, C.c_int32, dp, C.c_int32, dp, dp, dp, C.c_int32, C.c_double, C.c_double,
                                C.c_double, C.c_double, C.POINTER(vp)]
    L.sb_load_bandpasses.restype = C.c_int
    L.sb_load_bandpasses.argtypes = [C.c_int32, C.POINTER(C.c_int64), dp, dp, C.POINTER(vp)]
    L.sb_free_model.argtypes = [vp]
    L.sb_free_model.restype = None
    L.sb_free_bands.argtypes = [vp]
    L.sb_free_bands.restype = None
    L.sb_bandflux.restype = C.c_int
    L.sb_bandflux.argtypes = [vp, vp, C.POINTER(_Batch), vp, vp]
    L.sb_chi2.restype = C.c_int
    L.sb_chi2.argtypes = [vp, vp, C.POINTER(_Batch), vp, vp, vp, vp, vp]
    L.sb_chi2_noalloc.restype = C.c_int
    L.sb_chi2_noalloc.argtypes = [vp, vp, C.POINTER(_Batch), vp, vp, vp, vp, vp]
    L.sb_bandflux_grad.restype = C.c_int
    L.sb_bandflux_grad.argtypes = [vp, vp, C.POINTER(_Batch), vp, vp, vp, vp, vp, vp, vp]
    L.sb_pack_observations.restype = C.c_int
    L.sb_pack_observations.argtypes = [vp, vp, C.POINTER(_Batch), vp, C.POINTER(vp)]
    L.sb_free_pack.argtypes = [vp]
    L.sb_free_pack.restype = None
    L.sb_chi2_host.restype = C.c_int
    L.sb_chi2_host.argtypes = [vp, vp, C.POINTER(_Batch), vp, vp, vp, vp]
    L.sb_bandflux_grad_host.restype = C.c_int
    L.sb_bandflux_grad_host.argtypes = [vp, vp, C.POINTER(_Batch), vp, vp, vp, vp, vp, vp]
    L.sb_fit_default_opts.restype = None
    L.sb_fit_default_opts.argtypes = [C.POINTER(_FitOpts)]
    L.sb_fit_lbfgs.restype = C.c_int
    L.sb_fit_lbfgs.argtypes = [vp, vp, C.POINTER(_Batch), vp, vp, C.POINTER(_FitOpts), C.POINTER(_FitResult), vp]
    L.sb_fit_lbfgs_host.restype = C.c_int
    L.sb_fit_lbfgs_host.argtypes = [vp, vp, C.POINTER(_Batch), vp, vp, C.POINTER(_FitOpts), C.POINTER(_FitResult)]
    L.sb_bands_count.restype = C.c_int32
    L.sb_bands_count.argtypes = [vp]
    L.sb_bands_zpab.restype = C.c_double
    L.sb_bands_zpab.argtypes = [vp, C.c_int32]
    L.sb_last_launch_count.restype = C.c_int32
    L.sb_last_cuda_error.restype = C.c_int32
    L.sb_last_form.restype = C.c_int32
    L.sb_strerror.restype = C.c_char_p
    L.sb_strerror.argtypes = [C.c_int]
    L.sb_version.restype = C.c_char_p
    _lib = L
    return L


def _check(rc: int, what: str) -> None:
    if rc != 0:
        L = _load()
        msg = L.sb_strerror(rc).decode()
        raise SaltbandError(f"{what}: {msg} (status {rc}, cudaError {L.sb_last_cuda_error()})")


def version() -> str:
    return _load().sb_version().decode()


def last_launch_count() -> int:
    return int(_load().sb_last_launch_count())


def last_form() -> str:
    """Formulation the most recent compute call ran: 'direct', 'grouped', 'tiled' or ''."""
    return {SB_FORM_DIRECT: "direct", SB_FORM_GROUPED: "grouped", SB_FORM_TILED: "tiled"}.get(int(_load().sb_last_form()), "")


def _f64(a) -> np.ndarray:
    return np.ascontiguousarray(np.asarray(a, dtype=np.float64))


def _dptr(a: np.ndarray):
    return a.ctypes.data_as(C.POINTER(C.c_double))


class Model:
    """Owner of an `sb_model*` (device-resident M0/M1 tables and colour law)."""

    def __init__(self, handle: int):
        self._h = C.c_void_p(handle)

    def __del__(self):
        h, self._h = getattr(self, "_h", None), None
        if h and _lib is not None:
            _lib.sb_free_model(h)


class Bands:
    """Owner of an `sb_bands*` (device-resident band tables, folded weights, ZPAB)."""

    def __init__(self, handle: int):
        self._h = C.c_void_p(handle)

    def __del__(self):
        h, self._h = getattr(self, "_h", None), None
        if h and _lib is not None:
            _lib.sb_free_bands(h)

    @property
    def n_bands(self) -> int:
        return int(_load().sb_bands_count(self._h))

    def zpab(self, band: int) -> float:
        return float(_load().sb_bands_zpab(self._h, band))


class Pack:
    """Owner of an `sb_pack*` (theta-independent precompute of one batch: redshift order, item geometry)."""

    def __init__(self, handle: int, keep):
        self._h = C.c_void_p(handle)
        self._keep = keep  # the model and bands handles (and z) must outlive the pack

    def __del__(self):
        h, self._h = getattr(self, "_h", None), None
        if h and _lib is not None:
            _lib.sb_free_pack(h)


def sb_load_model(phase, wave, m0, m1, cl_coef, cl_wave_b, cl_wave_v, cl_lo, cl_hi) -> Model:
    """include/saltband.h: sb_load_model.  Host fp64 arrays; m0/m1 are [n_phase][n_wave]."""
    L = _load()
    phase, wave, m0, m1, cl = _f64(phase), _f64(wave), _f64(m0), _f64(m1), _f64(cl_coef)
    if m0.shape != (len(phase), len(wave)) or m1.shape != m0.shape:
        raise ValueError("m0/m1 must be [n_phase][n_wave]")
    out = C.c_void_p()
    rc = L.sb_load_model(_dptr(phase), len(phase), _dptr(wave), len(wave), _dptr(m0), _dptr(m1), _dptr(cl),
                         len(cl), float(cl_wave_b), float(cl_wave_v), float(cl_lo), float(cl_hi), C.byref(out))
    _check(rc, "sb_load_model")
    return Model(out.value)


def sb_load_bandpasses(offset, wave, trans) -> Bands:
    """include/saltband.h: sb_load_bandpasses.  CSR-packed host arrays."""
    L = _load()
    offset = np.ascontiguousarray(np.asarray(offset, dtype=np.int64))
    wave, trans = _f64(wave), _f64(trans)
    if len(wave) != len(trans) or len(offset) < 2 or int(offset[-1]) != len(wave):
        raise ValueError("offset/wave/trans are inconsistent")
    out = C.c_void_p()
    rc = L.sb_load_bandpasses(len(offset) - 1, offset.ctypes.data_as(C.POINTER(C.c_int64)), _dptr(wave),
                              _dptr(trans), C.byref(out))
    _check(rc, "sb_load_bandpasses")
    return Bands(out.value)


def _ptr(t, dtype, n: Optional[int], name: str, allow_none: bool = False):
    import torch

    if t is None:
        if allow_none:
            return None
        raise ValueError(f"{name} is required")
    if not isinstance(t, torch.Tensor) or not t.is_cuda:
        raise ValueError(f"{name} must be a CUDA torch tensor (there is no CPU path)")
    if t.dtype != dtype:
        raise ValueError(f"{name} must have dtype {dtype}, got {t.dtype}")
    if not t.is_contiguous():
        raise ValueError(f"{name} must be contiguous")
    if n is not None and t.numel() != n:
        raise ValueError(f"{name} must have {n} elements, got {t.numel()}")
    return t.data_ptr()


def _batch(dtype: int, n_sn: int, n_samples: int, obs_offset, time, band, zp, z, x0, x1, c, t0,
           n_obs_total: int, pack=None):
    import torch

    ft = torch.float32 if (dtype & 0xFF) == SB_F32 else torch.float64
    n_units = n_sn * n_samples
    if pack is not None and not isinstance(pack, Pack):
        raise ValueError("pack must be a Pack from sb_pack_observations")
    return _Batch(
        dtype, n_sn, n_samples, n_obs_total,
        _ptr(obs_offset, torch.int32, n_sn + 1, "obs_offset"),
        _ptr(time, ft, n_obs_total, "time"), _ptr(band, torch.int32, n_obs_total, "band"),
        _ptr(zp, ft, n_obs_total, "zp", allow_none=True), _ptr(z, ft, n_sn, "z"),
        _ptr(x0, ft, n_units, "x0"), _ptr(x1, ft, n_units, "x1"), _ptr(c, ft, n_units, "c"),
        _ptr(t0, ft, n_units, "t0"), pack._h if pack is not None else None)


def sb_pack_observations(model: Model, bands: Bands, *, dtype: int, n_sn: int, z) -> Pack:
    """include/saltband.h: sb_pack_observations.  z: [n_sn] CUDA fp32 tensor; built on the current stream."""
    import torch

    bt = _Batch(dtype, n_sn, 1, 0, None, None, None, None, _ptr(z, torch.float32, n_sn, "z"), None, None, None, None,
                None)
    out = C.c_void_p()
    rc = _load().sb_pack_observations(model._h, bands._h, C.byref(bt), _stream(), C.byref(out))
    _check(rc, "sb_pack_observations")
    return Pack(out.value, (model, bands, z))


def _stream() -> int:
    import torch

    return torch.cuda.current_stream().cuda_stream


def sb_bandflux(model: Model, bands: Bands, *, dtype: int, n_sn: int, n_samples: int, n_obs_total: int,
                obs_offset, time, band, zp, z, x0, x1, c, t0, out_flux, pack=None) -> None:
    """include/saltband.h: sb_bandflux.  out_flux: [n_obs_total*n_samples] CUDA tensor (written)."""
    import torch

    ft = torch.float32 if (dtype & 0xFF) == SB_F32 else torch.float64
    bt = _batch(dtype, n_sn, n_samples, obs_offset, time, band, zp, z, x0, x1, c, t0, n_obs_total, pack)
    rc = _load().sb_bandflux(model._h, bands._h, C.byref(bt), _ptr(out_flux, ft, n_obs_total * n_samples, "out_flux"),
                             _stream())
    _check(rc, "sb_bandflux")


def sb_chi2(model: Model, bands: Bands, *, dtype: int, n_sn: int, n_samples: int, n_obs_total: int,
            obs_offset, time, band, zp, z, x0, x1, c, t0, flux, fluxerr, out_chi2, out_flux=None,
            pack=None) -> None:
    """include/saltband.h: sb_chi2.  out_chi2: [n_sn*n_samples]; out_flux optional."""
    import torch

    ft = torch.float32 if (dtype & 0xFF) == SB_F32 else torch.float64
    bt = _batch(dtype, n_sn, n_samples, obs_offset, time, band, zp, z, x0, x1, c, t0, n_obs_total, pack)
    rc = _load().sb_chi2(model._h, bands._h, C.byref(bt), _ptr(flux, ft, n_obs_total, "flux"),
                         _ptr(fluxerr, ft, n_obs_total, "fluxerr"),
                         _ptr(out_chi2, ft, n_sn * n_samples, "out_chi2"),
                         _ptr(out_flux, ft, n_obs_total * n_samples, "out_flux", allow_none=True), _stream())
    _check(rc, "sb_chi2")


def sb_chi2_noalloc(model: Model, bands: Bands, *, dtype: int, n_sn: int, n_samples: int, n_obs_total: int,
                    obs_offset, time, band, zp, z, x0, x1, c, t0, flux, fluxerr, out_chi2, out_flux=None) -> None:
    """include/saltband.h: sb_chi2_noalloc -- sb_chi2 for a caller that must not allocate device memory (its
    GPU memory all belongs to another pool, or it cannot take cudaMalloc's synchronisation).  fp32 only, no
    pack, n_sn <= SB_NOALLOC_MAX_SN (SaltbandError 'table exceeds ...' beyond).  All calls on a device share
    one fixed scratch array inside the library: keep them ordered on the GPU (one stream, or events) -- calls
    that overlap there race.  The first call on a device also looks up that array's address; make it during
    set-up.  The tensors passed here are the caller's own, as for sb_chi2."""
    import torch

    if (dtype & 0xFF) != SB_F32:
        raise ValueError("sb_chi2_noalloc is fp32 only")
    ft = torch.float32
    bt = _batch(dtype, n_sn, n_samples, obs_offset, time, band, zp, z, x0, x1, c, t0, n_obs_total, None)
    rc = _load().sb_chi2_noalloc(model._h, bands._h, C.byref(bt), _ptr(flux, ft, n_obs_total, "flux"),
                                 _ptr(fluxerr, ft, n_obs_total, "fluxerr"),
                                 _ptr(out_chi2, ft, n_sn * n_samples, "out_chi2"),
                                 _ptr(out_flux, ft, n_obs_total * n_samples, "out_flux", allow_none=True), _stream())
    _check(rc, "sb_chi2_noalloc")


def sb_bandflux_grad(model: Model, bands: Bands, *, dtype: int, n_sn: int, n_samples: int, n_obs_total: int,
                     obs_offset, time, band, zp, z, x0, x1, c, t0, flux=None, fluxerr=None, out_flux=None,
                     out_dflux=None, out_chi2=None, out_dchi2=None, pack=None) -> None:
    """include/saltband.h: sb_bandflux_grad.  Gradient order: (x0, x1, c, t0)."""
    import torch

    ft = torch.float32 if (dtype & 0xFF) == SB_F32 else torch.float64
    bt = _batch(dtype, n_sn, n_samples, obs_offset, time, band, zp, z, x0, x1, c, t0, n_obs_total, pack)
    n_ev, n_units = n_obs_total * n_samples, n_sn * n_samples
    rc = _load().sb_bandflux_grad(
        model._h, bands._h, C.byref(bt), _ptr(flux, ft, n_obs_total, "flux", allow_none=True),
        _ptr(fluxerr, ft, n_obs_total, "fluxerr", allow_none=True),
        _ptr(out_flux, ft, n_ev, "out_flux", allow_none=True),
        _ptr(out_dflux, ft, n_ev * 4, "out_dflux", allow_none=True),
        _ptr(out_chi2, ft, n_units, "out_chi2", allow_none=True),
        _ptr(out_dchi2, ft, n_units * 4, "out_dchi2", allow_none=True), _stream())
    _check(rc, "sb_bandflux_grad")


# ---------------------------------------------------------------- host-buffer calls
def _hptr(t, dtype, n: Optional[int], name: str, allow_none: bool = False):
    """Host pointer of a CPU torch tensor (pinned or pageable) of the given dtype and size."""
    import torch

    if t is None:
        if allow_none:
            return None
        raise ValueError(f"{name} is required")
    if not isinstance(t, torch.Tensor) or t.is_cuda:
        raise ValueError(f"{name} must be a CPU torch tensor (pin it for the full PCIe rate)")
    if t.dtype != dtype or not t.is_contiguous():
        raise ValueError(f"{name} must be a contiguous tensor of dtype {dtype}")
    if n is not None and t.numel() != n:
        raise ValueError(f"{name} must have {n} elements, got {t.numel()}")
    return t.data_ptr()


def _host_batch(dtype, n_sn, n_samples, n_obs_total, obs_offset, time, band, zp, z, x0, x1, c, t0):
    import torch

    ft = torch.float32 if (dtype & 0xFF) == SB_F32 else torch.float64
    n_units = n_sn * n_samples
    return ft, _Batch(
        dtype, n_sn, n_samples, n_obs_total, _hptr(obs_offset, torch.int32, n_sn + 1, "obs_offset"),
        _hptr(time, ft, n_obs_total, "time"), _hptr(band, torch.int32, n_obs_total, "band"),
        _hptr(zp, ft, n_obs_total, "zp", allow_none=True), _hptr(z, ft, n_sn, "z"), _hptr(x0, ft, n_units, "x0"),
        _hptr(x1, ft, n_units, "x1"), _hptr(c, ft, n_units, "c"), _hptr(t0, ft, n_units, "t0"), None)


def sb_chi2_host(model: Model, bands: Bands, *, dtype: int, n_sn: int, n_samples: int, n_obs_total: int,
                 obs_offset, time, band, zp, z, x0, x1, c, t0, flux, fluxerr, out_chi2, out_flux=None) -> None:
    """include/saltband.h: sb_chi2_host.  Every array is a CPU tensor; returns when the outputs are complete."""
    ft, bt = _host_batch(dtype, n_sn, n_samples, n_obs_total, obs_offset, time, band, zp, z, x0, x1, c, t0)
    rc = _load().sb_chi2_host(model._h, bands._h, C.byref(bt), _hptr(flux, ft, n_obs_total, "flux"),
                              _hptr(fluxerr, ft, n_obs_total, "fluxerr"),
                              _hptr(out_chi2, ft, n_sn * n_samples, "out_chi2"),
                              _hptr(out_flux, ft, n_obs_total * n_samples, "out_flux", allow_none=True))
    _check(rc, "sb_chi2_host")


def sb_bandflux_grad_host(model: Model, bands: Bands, *, dtype: int, n_sn: int, n_samples: int, n_obs_total: int,
                          obs_offset, time, band, zp, z, x0, x1, c, t0, flux=None, fluxerr=None, out_flux=None,
                          out_dflux=None, out_chi2=None, out_dchi2=None) -> None:
    """include/saltband.h: sb_bandflux_grad_host.  Gradient order: (x0, x1, c, t0)."""
    ft, bt = _host_batch(dtype, n_sn, n_samples, n_obs_total, obs_offset, time, band, zp, z, x0, x1, c, t0)
    n_ev, n_units = n_obs_total * n_samples, n_sn * n_samples
    rc = _load().sb_bandflux_grad_host(
        model._h, bands._h, C.byref(bt), _hptr(flux, ft, n_obs_total, "flux", allow_none=True),
        _hptr(fluxerr, ft, n_obs_total, "fluxerr", allow_none=True),
        _hptr(out_flux, ft, n_ev, "out_flux", allow_none=True),
        _hptr(out_dflux, ft, n_ev * 4, "out_dflux", allow_none=True),
        _hptr(out_chi2, ft, n_units, "out_chi2", allow_none=True),
        _hptr(out_dchi2, ft, n_units * 4, "out_dchi2", allow_none=True))
    _check(rc, "sb_bandflux_grad_host")


# ---------------------------------------------------------------- batched L-BFGS fit
def _fit_opts(memory, max_eval, max_iter, trace_len, ftol, gtol, lo, hi):
    """sb_fit_opts with the library's defaults (sb_fit_default_opts) for every argument left None."""
    o = _FitOpts()
    _load().sb_fit_default_opts(C.byref(o))
    keep = []
    for name, v in (("memory", memory), ("max_eval", max_eval), ("max_iter", max_iter), ("trace_len", trace_len),
                    ("ftol", ftol), ("gtol", gtol)):
        if v is not None:
            setattr(o, name, v)
    for name, v in (("lo", lo), ("hi", hi)):
        if v is not None:
            arr = _f64(v)
            if arr.shape != (4,):
                raise ValueError(f"{name} must have 4 elements (x0, x1, c, t0)")
            keep.append(arr)
            setattr(o, name, _dptr(arr))
    return o, keep


def sb_fit_lbfgs(model: Model, bands: Bands, *, dtype: int, n_sn: int, n_samples: int, n_obs_total: int,
                 obs_offset, time, band, zp, z, x0, x1, c, t0, flux, fluxerr, out_theta, out_chi2, out_status=None,
                 out_n_iter=None, out_n_eval=None, out_trace=None, pack=None, memory=None, max_eval=None,
                 max_iter=None, ftol=None, gtol=None, lo=None, hi=None) -> None:
    """include/saltband.h: sb_fit_lbfgs.  x0, x1, c, t0 are the start point; every array is a CUDA tensor; the
    fit is enqueued on the current stream (no synchronisation).  out_trace: [trace_len, n_units] fp64."""
    import torch

    ft = torch.float32 if (dtype & 0xFF) == SB_F32 else torch.float64
    n_units = n_sn * n_samples
    bt = _batch(dtype, n_sn, n_samples, obs_offset, time, band, zp, z, x0, x1, c, t0, n_obs_total, pack)
    trace_len = 0 if out_trace is None else out_trace.shape[0]
    opts, keep = _fit_opts(memory, max_eval, max_iter, trace_len, ftol, gtol, lo, hi)
    res = _FitResult(_ptr(out_theta, ft, 4 * n_units, "out_theta"), _ptr(out_chi2, ft, n_units, "out_chi2"),
                     _ptr(out_status, torch.int32, n_units, "out_status", allow_none=True),
                     _ptr(out_n_iter, torch.int32, n_units, "out_n_iter", allow_none=True),
                     _ptr(out_n_eval, torch.int32, n_units, "out_n_eval", allow_none=True),
                     _ptr(out_trace, torch.float64, trace_len * n_units, "out_trace", allow_none=True))
    rc = _load().sb_fit_lbfgs(model._h, bands._h, C.byref(bt), _ptr(flux, ft, n_obs_total, "flux"),
                              _ptr(fluxerr, ft, n_obs_total, "fluxerr"), C.byref(opts), C.byref(res), _stream())
    del keep
    _check(rc, "sb_fit_lbfgs")


def sb_fit_lbfgs_host(model: Model, bands: Bands, *, dtype: int, n_sn: int, n_samples: int, n_obs_total: int,
                      obs_offset, time, band, zp, z, x0, x1, c, t0, flux, fluxerr, out_theta, out_chi2,
                      out_status=None, out_n_iter=None, out_n_eval=None, out_trace=None, memory=None, max_eval=None,
                      max_iter=None, ftol=None, gtol=None, lo=None, hi=None) -> None:
    """include/saltband.h: sb_fit_lbfgs_host.  Every array is a CPU tensor; returns when the results are complete."""
    import torch

    ft, bt = _host_batch(dtype, n_sn, n_samples, n_obs_total, obs_offset, time, band, zp, z, x0, x1, c, t0)
    n_units = n_sn * n_samples
    trace_len = 0 if out_trace is None else out_trace.shape[0]
    opts, keep = _fit_opts(memory, max_eval, max_iter, trace_len, ftol, gtol, lo, hi)
    res = _FitResult(_hptr(out_theta, ft, 4 * n_units, "out_theta"), _hptr(out_chi2, ft, n_units, "out_chi2"),
                     _hptr(out_status, torch.int32, n_units, "out_status", allow_none=True),
                     _hptr(out_n_iter, torch.int32, n_units, "out_n_iter", allow_none=True),
                     _hptr(out_n_eval, torch.int32, n_units, "out_n_eval", allow_none=True),
                     _hptr(out_trace, torch.float64, trace_len * n_units, "out_trace", allow_none=True))
    rc = _load().sb_fit_lbfgs_host(model._h, bands._h, C.byref(bt), _hptr(flux, ft, n_obs_total, "flux"),
                                   _hptr(fluxerr, ft, n_obs_total, "fluxerr"), C.byref(opts), C.byref(res))
    del keep
    _check(rc, "sb_fit_lbfgs_host")
