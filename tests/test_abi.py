"""CPU-side checks of the C ABI: libmlens.so loads, exports every symbol include/mlens.h declares, validates its
arguments before touching CUDA, and fails loudly (no CPU fallback) when there is no device."""
import ctypes
import os
import re

import numpy as np
import pytest

from paper_1406_0559_b200 import mlens

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def L():
    from paper_1406_0559_b200 import build

    build.build()
    return mlens.lib()


def test_every_declared_symbol_is_exported(L):
    header = open(os.path.join(ROOT, "include", "mlens.h")).read()
    header = re.sub(r"/\*.*?\*/", "", header, flags=re.S)
    names = set(re.findall(r"\b(mlens_[a-z_]+)\s*\(", header))
    assert {"mlens_create", "mlens_shoot", "mlens_destroy", "mlens_shoot_block", "mlens_get_geometry",
            "mlens_last_error"} <= names
    for n in names:
        assert hasattr(L, n), n


def _create(L, kappa=0.3, gamma=0.2, s=0.0, side=4.0, npix=64, d=0.01, xy=None, m=None, n=None):
    h = ctypes.c_void_p()
    xy = np.zeros(2, np.float32) if xy is None else np.asarray(xy, np.float32)
    n = xy.size // 2 if n is None else n
    rc = L.mlens_create(ctypes.byref(h), kappa, gamma, s, side, npix, d, xy.ctypes.data_as(ctypes.c_void_p),
                        None if m is None else np.asarray(m, np.float32).ctypes.data_as(ctypes.c_void_p), n)
    return rc, h


@pytest.mark.parametrize("kw", [
    dict(kappa=float("nan")), dict(kappa=-0.1), dict(s=1.5), dict(s=-0.1), dict(side=0.0), dict(npix=0), dict(d=0.0),
    dict(d=-1.0), dict(n=-1), dict(kappa=0.8, gamma=0.2),  # 1-kappa-gamma = 0: critical line
    dict(kappa=1.2, gamma=0.2),                             # 1-kappa+gamma = 0
    dict(xy=[0.0, float("inf")]), dict(xy=[0.0, 1.0], m=[0.0]), dict(xy=[0.0, 1.0], m=[-1.0]),
    dict(xy=[0.0, 1.0], m=[float("nan")]),
])
def test_create_rejects_bad_arguments(L, kw):
    rc, h = _create(L, **kw)
    assert rc == mlens.EINVAL and not h
    assert len(L.mlens_last_error()) > 0


def test_create_range_errors(L):
    rc, h = _create(L, npix=50000)  # npix^2 >= 2^31
    assert rc == mlens.ERANGE and not h
    rc, h = _create(L, d=1e-10)  # >= 2^31 rays along an axis
    assert rc == mlens.ERANGE and not h


def test_null_handles_are_rejected_not_crashing(L):
    assert L.mlens_shoot(None, None, None, None, None) == mlens.EINVAL
    assert L.mlens_shoot_block(None, 0, 0, 1, 1, None, None, None, None) == mlens.EINVAL
    assert L.mlens_get_geometry(None, None) == mlens.EINVAL
    assert L.mlens_set_option(None, b"kernel", 1) == mlens.EINVAL
    L.mlens_destroy(None)


def test_no_cpu_fallback_without_a_device(L):
    import torch

    if torch.cuda.is_available():
        pytest.skip("a CUDA device is present")
    rc, h = _create(L)
    assert rc == mlens.ECUDA and not h
    with pytest.raises(mlens.MlensError):
        mlens.Mlens(0.3, 0.2, 0.0, 4.0, 64, 0.01, np.zeros((1, 2), np.float32))
