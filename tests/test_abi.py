"""CPU-side checks of the boundary: the C-ABI library builds, loads, and exports every symbol that
include/saltband.h declares; host-side argument validation works without a GPU (no compute)."""
import ctypes as C
import os
import re

import numpy as np
import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
HEADER = os.path.join(ROOT, "include", "saltband.h")


@pytest.fixture(scope="module")
def lib():
    from paper_2504_08081_b200 import build as sbbuild
    from paper_2504_08081_b200 import api

    sbbuild.build()
    return api._load()


def _declared_functions():
    src = open(HEADER).read()
    src = re.sub(r"/\*.*?\*/", "", src, flags=re.S)
    names = set(re.findall(r"\b(sb_[a-z0-9_]+)\s*\(", src))
    return sorted(names)


def test_header_declares_the_five_north_star_calls():
    names = _declared_functions()
    for n in ("sb_load_model", "sb_load_bandpasses", "sb_bandflux", "sb_chi2", "sb_bandflux_grad"):
        assert n in names


def test_library_exports_every_declared_symbol(lib):
    for n in _declared_functions():
        assert hasattr(lib, n), f"libsaltband.so does not export {n}"


def test_no_torch_types_in_the_abi():
    src = open(HEADER).read()
    assert "torch" not in src.lower().replace("torch tensors", "") and "at::" not in src and "c10::" not in src


def test_strerror_and_version(lib):
    assert lib.sb_strerror(0) == b"ok"
    assert b"invalid" in lib.sb_strerror(-1)
    assert b"sm_100a" in lib.sb_version()


def test_loader_argument_validation_is_host_side(lib):
    """Bad grids are rejected with SB_EINVAL before any CUDA call (so this runs without a GPU)."""
    dp = C.POINTER(C.c_double)
    phase = np.array([0.0, 1.0, 2.5])  # non-uniform
    wave = np.array([1000.0, 1010.0, 1020.0])
    m = np.zeros((3, 3))
    cl = np.zeros(5)
    out = C.c_void_p()
    p = lambda a: a.ctypes.data_as(dp)
    rc = lib.sb_load_model(p(phase), 3, p(wave), 3, p(m), p(m), p(cl), 5, 4302.57, 5428.55, 2800.0, 7000.0, C.byref(out))
    assert rc == -1 and not out.value
    phase = np.array([0.0, 1.0, 2.0])
    m_bad = m.copy()
    m_bad[1, 1] = np.nan
    rc = lib.sb_load_model(p(phase), 3, p(wave), 3, p(m_bad), p(m), p(cl), 5, 4302.57, 5428.55, 2800.0, 7000.0, C.byref(out))
    assert rc == -1
    rc = lib.sb_load_model(p(phase), 3, p(wave), 3, p(m), p(m), p(cl), 9, 4302.57, 5428.55, 2800.0, 7000.0, C.byref(out))
    assert rc == -1  # n_cl > 8
    off = np.array([0, 3], dtype=np.int64)
    w_bad = np.array([5000.0, 4990.0, 5010.0])
    t = np.ones(3)
    rc = lib.sb_load_bandpasses(1, off.ctypes.data_as(C.POINTER(C.c_int64)), p(w_bad), p(t), C.byref(out))
    assert rc == -1 and not out.value
    off1 = np.array([0, 1], dtype=np.int64)
    rc = lib.sb_load_bandpasses(1, off1.ctypes.data_as(C.POINTER(C.c_int64)), p(w_bad), p(t), C.byref(out))
    assert rc == -1  # < 2 points


def test_compute_call_null_arguments(lib):
    assert lib.sb_bandflux(None, None, None, None, None) == -1
    assert lib.sb_chi2(None, None, None, None, None, None, None, None) == -1
    assert lib.sb_last_launch_count() == 0


def test_binding_rejects_cpu_tensors():
    import torch

    import paper_2504_08081_b200 as sb
    from paper_2504_08081_b200 import api

    with pytest.raises(ValueError):
        api._ptr(torch.zeros(3), torch.float32, 3, "x")
    assert os.path.basename(sb.lib_path()) == "libsaltband.so"


def test_product_does_not_import_oracle():
    pkg = os.path.join(ROOT, "paper_2504_08081_b200")
    for dirpath, _, files in os.walk(pkg):
        for f in files:
            if f.endswith((".py", ".cu", ".cuh", ".h")):
                txt = open(os.path.join(dirpath, f)).read()
                assert "import oracle" not in txt and "from oracle" not in txt and "salt_oracle" not in txt
    for f in os.listdir(os.path.join(ROOT, "oracle")):
        if f.endswith((".py", ".c")):
            txt = open(os.path.join(ROOT, "oracle", f)).read()
            assert "import paper_2504_08081_b200" not in txt and "saltband.h\"" not in txt


def test_fit_options_defaults_and_host_side_validation(lib):
    """sb_fit_default_opts fills the documented defaults; sb_fit_lbfgs rejects NULL handles, missing
    photometry and out-of-range options with SB_EINVAL before any CUDA call (runs without a GPU)."""
    from paper_2504_08081_b200 import api

    o = api._FitOpts()
    lib.sb_fit_default_opts(C.byref(o))
    assert (o.memory, o.max_eval, o.max_iter, o.trace_len) == (8, 60, 1000, 0)
    assert o.ftol == 1e-12 and o.gtol == 0.0 and not o.lo and not o.hi
    bt = api._Batch(api.SB_F32, 1, 1, 0, None, None, None, None, None, None, None, None, None, None)
    res = api._FitResult(None, None, None, None, None, None)
    assert lib.sb_fit_lbfgs(None, None, C.byref(bt), None, None, C.byref(o), C.byref(res), None) == -1
    assert lib.sb_fit_lbfgs_host(None, None, C.byref(bt), None, None, C.byref(o), C.byref(res)) == -1
    assert lib.sb_pack_observations(None, None, C.byref(bt), None, C.byref(C.c_void_p())) == -1
    lib.sb_free_pack(None)  # NULL is allowed


def test_binding_exposes_the_same_names_as_the_header():
    import paper_2504_08081_b200 as sb

    for n in ("sb_load_model", "sb_load_bandpasses", "sb_bandflux", "sb_chi2", "sb_bandflux_grad", "sb_pack_observations",
              "sb_fit_lbfgs", "sb_chi2_host", "sb_bandflux_grad_host", "sb_fit_lbfgs_host"):
        assert callable(getattr(sb, n)), n
