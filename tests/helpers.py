"""Glue shared by the tests: Workload -> oracle.Problem, error norms."""
import numpy as np

import oracle


def problem(wl, **over):
    kw = dict(nz=wl.nz, nx=wl.nx, dx=wl.dx, dt=wl.dt, nt=wl.nt, npml=wl.npml, pml_order=wl.pml_order,
              pml_sigma_max=wl.pml_sigma_max, pml_kappa_max=wl.pml_kappa_max,
              pml_alpha_max=wl.pml_alpha_max, src_zx=wl.src_zx, rec_zx=wl.rec_zx,
              wavelet=wl.wavelet.astype(np.float64))
    kw.update(over)
    return oracle.Problem(**kw)


def rel_l2(a, b):
    a = np.asarray(a, dtype=np.float64)
    b = np.asarray(b, dtype=np.float64)
    return float(np.linalg.norm((a - b).ravel()) / max(np.linalg.norm(b.ravel()), 1e-300))
