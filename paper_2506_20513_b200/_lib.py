"""ctypes view of libgprfwi.so (include/gprfwi.h).  Argument marshalling only.

The library is built in-tree by ``build.py`` (nvcc, sm_100a).  There is NO fallback: if the shared
library is missing, ``load()`` raises.
"""
from __future__ import annotations

import ctypes
import os

_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(_HERE, "libgprfwi.so")

GPRFWI_OK = 0
STATUS_NAMES = {0: "OK", -1: "EINVAL", -2: "ECFL", -3: "EGEOM", -4: "ENOMEM", -5: "ESTATE", -6: "ECUDA", -7: "ETOOBIG"}

EXPORTS = (
    "gprfwi_workspace_bytes", "gprfwi_forward", "gprfwi_forward_mu", "gprfwi_adjoint", "gprfwi_gradient_host",
    "gprfwi_workspace_bytes_host", "gprfwi_residual", "gprfwi_launch_count", "gprfwi_get_plan",
    "gprfwi_release", "gprfwi_strerror", "gprfwi_version", "gprfwi_update", "gprfwi_update_workspace_bytes", "gprfwi_lowpass",
    "gprfwi_lowpass_design", "gprfwi_restrict", "gprfwi_prolong_add",
    "gprfwi_update_noalloc", "gprfwi_update_noalloc_max_bytes",
)


class Params(ctypes.Structure):
    """gprfwi_params"""
    _fields_ = [
        ("nz", ctypes.c_int32), ("nx", ctypes.c_int32), ("pitch", ctypes.c_int32),
        ("dx", ctypes.c_float), ("dt", ctypes.c_float), ("nt", ctypes.c_int32),
        ("npml", ctypes.c_int32), ("pml_order", ctypes.c_int32),
        ("pml_sigma_max", ctypes.c_float), ("pml_kappa_max", ctypes.c_float),
        ("pml_alpha_max", ctypes.c_float),
        ("nshots", ctypes.c_int32), ("nrec", ctypes.c_int32),
        ("wavelet_per_shot", ctypes.c_int32), ("checkpoint_stride", ctypes.c_int32),
    ]


class Plan(ctypes.Structure):
    """gprfwi_plan"""
    _fields_ = [
        ("workspace_bytes", ctypes.c_uint64), ("full_history", ctypes.c_int32),
        ("checkpoint_stride", ctypes.c_int32), ("shots_per_pass", ctypes.c_int32),
        ("time_block", ctypes.c_int32), ("stored_segments", ctypes.c_int32), ("reserved", ctypes.c_int32),
    ]

    def as_dict(self):
        return {k: int(getattr(self, k)) for k, _ in self._fields_}


class UpdateParams(ctypes.Structure):
    """gprfwi_update_params"""
    _fields_ = [
        ("step", ctypes.c_int32), ("lr_eps_r", ctypes.c_float), ("lr_sigma", ctypes.c_float),
        ("beta1", ctypes.c_float), ("beta2", ctypes.c_float), ("adam_eps", ctypes.c_float),
        ("tv_iters", ctypes.c_int32), ("tv_rho", ctypes.c_float), ("tv_lambda", ctypes.c_float),
        ("tv_alpha", ctypes.c_float), ("mask_rows", ctypes.c_int32),
        ("eps_r_min", ctypes.c_float), ("sigma_min", ctypes.c_float),
    ]


class GprfwiError(RuntimeError):
    def __init__(self, code, text):
        super().__init__(f"gprfwi: {STATUS_NAMES.get(code, code)}: {text}")
        self.code = code


_lib = None


def _declare(lib):
    vp, sz, i32p, fp = ctypes.c_void_p, ctypes.c_size_t, ctypes.c_void_p, ctypes.c_void_p
    lib.gprfwi_workspace_bytes.restype = sz
    lib.gprfwi_workspace_bytes.argtypes = [ctypes.POINTER(Params), sz, ctypes.POINTER(Plan)]
    lib.gprfwi_workspace_bytes_host.restype = sz
    lib.gprfwi_workspace_bytes_host.argtypes = [ctypes.POINTER(Params), sz]
    lib.gprfwi_forward.restype = ctypes.c_int
    lib.gprfwi_forward.argtypes = [ctypes.POINTER(vp), ctypes.POINTER(Params), fp, fp, fp, i32p, i32p,
                                   vp, sz, fp, vp]
    lib.gprfwi_forward_mu.restype = ctypes.c_int
    lib.gprfwi_forward_mu.argtypes = [ctypes.POINTER(vp), ctypes.POINTER(Params), fp, fp, fp, fp, i32p, i32p,
                                      vp, sz, fp, vp]
    lib.gprfwi_adjoint.restype = ctypes.c_int
    lib.gprfwi_adjoint.argtypes = [vp, fp, fp, fp, vp]
    lib.gprfwi_gradient_host.restype = ctypes.c_int
    lib.gprfwi_gradient_host.argtypes = [ctypes.POINTER(Params), fp, fp, fp, i32p, i32p, fp, vp, sz,
                                         fp, fp, fp, ctypes.POINTER(ctypes.c_double), vp]
    lib.gprfwi_residual.restype = ctypes.c_int
    lib.gprfwi_residual.argtypes = [fp, fp, fp, sz, vp, vp]
    lib.gprfwi_launch_count.restype = ctypes.c_int64
    lib.gprfwi_launch_count.argtypes = [vp]
    lib.gprfwi_get_plan.restype = ctypes.c_int
    lib.gprfwi_get_plan.argtypes = [vp, ctypes.POINTER(Plan)]
    lib.gprfwi_release.restype = None
    lib.gprfwi_release.argtypes = [vp]
    lib.gprfwi_strerror.restype = ctypes.c_char_p
    lib.gprfwi_strerror.argtypes = [ctypes.c_int]
    lib.gprfwi_update_workspace_bytes.restype = sz
    lib.gprfwi_update_workspace_bytes.argtypes = [ctypes.c_int32, ctypes.c_int32]
    lib.gprfwi_update.restype = ctypes.c_int
    lib.gprfwi_update.argtypes = [ctypes.c_int32, ctypes.c_int32, ctypes.c_int32, ctypes.POINTER(UpdateParams),
                                  fp, fp, fp, fp, fp, fp, fp, fp, vp, sz, vp]
    lib.gprfwi_lowpass.restype = ctypes.c_int
    lib.gprfwi_lowpass.argtypes = [fp, fp, ctypes.c_int32, ctypes.c_int32, ctypes.c_int32, fp, ctypes.c_int32, vp]
    lib.gprfwi_lowpass_design.restype = ctypes.c_int32
    lib.gprfwi_lowpass_design.argtypes = [ctypes.c_float, ctypes.c_float, ctypes.c_int32, fp]
    lib.gprfwi_restrict.restype = ctypes.c_int
    lib.gprfwi_restrict.argtypes = [fp, ctypes.c_int32, ctypes.c_int32, ctypes.c_int32, fp, ctypes.c_int32, vp]
    lib.gprfwi_prolong_add.restype = ctypes.c_int
    lib.gprfwi_prolong_add.argtypes = [fp, ctypes.c_int32, ctypes.c_float, fp, ctypes.c_int32, ctypes.c_int32,
                                       ctypes.c_int32, vp]
    lib.gprfwi_update_noalloc.restype = ctypes.c_int
    lib.gprfwi_update_noalloc.argtypes = [ctypes.c_int32, ctypes.c_int32, ctypes.c_int32, ctypes.POINTER(UpdateParams),
                                          fp, fp, fp, fp, fp, fp, fp, fp, vp]
    lib.gprfwi_update_noalloc_max_bytes.restype = sz
    lib.gprfwi_update_noalloc_max_bytes.argtypes = []
    lib.gprfwi_version.restype = ctypes.c_int
    return lib


def load():
    """Load the in-tree CUDA library; fail loudly if it has not been built."""
    global _lib
    if _lib is None:
        if not os.path.exists(LIB_PATH):
            raise ImportError(
                f"{LIB_PATH} is missing: run `python -m paper_2506_20513_b200.build` "
                "(there is no CPU fallback)")
        _lib = _declare(ctypes.CDLL(LIB_PATH))
    return _lib


def check(code):
    if code != GPRFWI_OK:
        raise GprfwiError(code, load().gprfwi_strerror(code).decode())
