"""CPU-side checks of the C-ABI library: it builds for sm_100a, loads without a GPU, exports every
symbol include/ak.h declares, and validates arguments before touching CUDA."""
import ctypes as C
import os
import re

import numpy as np
import pytest

from paper_2409_10384_b200 import ak, build

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def lib():
    build.build()
    return ak.lib()


def declared_symbols():
    src = open(os.path.join(ROOT, "include", "ak.h")).read()
    src = re.sub(r"/\*.*?\*/", "", src, flags=re.S)
    return sorted(set(re.findall(r"\b(ak_[a-z0-9_]+)\s*\(", src)))


def test_header_symbols_are_exported(lib):
    names = declared_symbols()
    assert len(names) >= 12 and "ak_rhs" in names and "ak_con2prim" in names and "ak_emf" in names
    for nm in names:
        assert hasattr(lib, nm), "libak.so does not export %s" % nm
    assert set(names) == set(ak.EXPORTS)


def test_version_and_strerror(lib):
    assert "sm_100a" in ak.version()
    assert ak.strerror(0) == "ok"
    assert "invalid" in ak.strerror(ak.AK_EINVAL)


def good_params(**kw):
    p = dict(nmb=1, n=8, gamma_ad=2.0, rho_atm=1e-10, T_atm=1e-8)
    p.update(kw)
    return ak.make_params(**p)


@pytest.mark.parametrize("bad", [dict(n=1), dict(ng=3), dict(gamma_ad=1.0), dict(rho_atm=-1.0), dict(T_atm=0.0),
                                 dict(f_thr=float("nan")), dict(mag_max=0.0), dict(recon=5), dict(riemann=2),
                                 dict(fofc=2), dict(dmp_M=0.5), dict(c2p_max_iter=0), dict(c2p_tol=0.0),
                                 dict(device=-1), dict(nmb=0), dict(nmb=40000, n=32)])
def test_create_rejects_bad_params_before_cuda(lib, bad):
    p = good_params(**bad)
    dx = np.full((max(p.nmb, 1), 3), 0.1)
    h = C.c_void_p()
    assert lib.ak_create(C.byref(p), dx.ctypes.data_as(C.POINTER(C.c_double)), C.byref(h)) == ak.AK_EINVAL
    assert not h.value


def test_create_rejects_bad_dx_and_null(lib):
    p = good_params()
    dx = np.array([[0.1, -0.1, 0.1]])
    h = C.c_void_p()
    assert lib.ak_create(C.byref(p), dx.ctypes.data_as(C.POINTER(C.c_double)), C.byref(h)) == ak.AK_EINVAL
    assert lib.ak_create(None, dx.ctypes.data_as(C.POINTER(C.c_double)), C.byref(h)) == ak.AK_EINVAL
    assert lib.ak_create(C.byref(p), None, C.byref(h)) == ak.AK_EINVAL
    assert lib.ak_destroy(None) == ak.AK_EINVAL
    assert lib.ak_rhs(None, None, None, None, 0, 0.1, None) == ak.AK_EINVAL


def test_no_gpu_means_error_not_fallback(lib):
    """Without a CUDA device ak_create must fail (AK_ECUDA / AK_EINVAL), never succeed on the CPU."""
    import torch
    if torch.cuda.is_available():
        pytest.skip("GPU present")
    p = good_params()
    dx = np.full((1, 3), 0.1)
    with pytest.raises(ak.AkError):
        ak.ak_create(p, dx)


def test_product_does_not_import_oracle():
    pk = os.path.join(ROOT, "paper_2409_10384_b200")
    for dp, _, fs in os.walk(pk):
        for f in fs:
            if f.endswith((".py", ".cu", ".cuh", ".h")):
                s = open(os.path.join(dp, f)).read()
                assert "pyoracle" not in s and "oracle.h" not in s and "liboracle" not in s, f
