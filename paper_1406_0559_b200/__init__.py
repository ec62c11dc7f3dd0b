"""mlens — B200-native (sm_100a) direct inverse ray-shooting for quasar-microlensing magnification maps.

Hot path of GERLUMPH / GPU-D (Vernardos & Fluke 2014, arXiv:1406.0559, Eq. 1 and Eq. 4).  The compute path is the
C-ABI library ``libmlens.so`` (``include/mlens.h``); this package is a thin binding (``mlens``) plus the seeded input
generators (``fields``).  There is no CPU fallback: using the binding without the built CUDA library raises.
"""
from . import fields  # noqa: F401  (pure numpy; safe without a GPU)

__all__ = ["fields", "mlens"]


def __getattr__(name):
    if name == "mlens":
        import importlib

        return importlib.import_module(".mlens", __name__)
    raise AttributeError(name)
