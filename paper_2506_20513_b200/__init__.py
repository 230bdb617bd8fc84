"""B200-native forward + exact-adjoint 2-D TM FDTD for GPR dual-parameter FWI (arxiv/paper_2506_20513).

Thin Python binding over the C-ABI library ``libgprfwi.so`` (include/gprfwi.h).  PyTorch is used only
for device memory and streams; every step of the path runs in the library's CUDA kernels.
"""
from ._lib import GprfwiError, Params, Plan, UpdateParams, EXPORTS, LIB_PATH  # noqa: F401
from .api import (Simulation, Stage, split_batch, invert, invert_staged, gprfwi_lowpass, gprfwi_lowpass_design, gprfwi_restrict, gprfwi_prolong_add, coarse_problem, gprfwi_adjoint, gprfwi_forward, gprfwi_gradient_host,  # noqa: F401
                  gprfwi_residual, gprfwi_update, gprfwi_update_noalloc, gprfwi_update_noalloc_max_bytes,
                  gprfwi_update_workspace_bytes, gprfwi_workspace_bytes,
                  gprfwi_workspace_bytes_host, make_params, make_update_params)

__all__ = ["Simulation", "Stage", "split_batch", "invert", "invert_staged", "gprfwi_lowpass", "gprfwi_lowpass_design", "gprfwi_restrict", "gprfwi_prolong_add", "coarse_problem", "make_params", "gprfwi_workspace_bytes", "gprfwi_workspace_bytes_host",
           "gprfwi_forward", "gprfwi_adjoint", "gprfwi_gradient_host", "gprfwi_residual",
           "gprfwi_update", "gprfwi_update_noalloc", "gprfwi_update_noalloc_max_bytes", "gprfwi_update_workspace_bytes", "make_update_params",
           "GprfwiError", "Params", "Plan", "UpdateParams"]
