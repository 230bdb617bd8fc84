"""Float64 CPU oracle for the GPR-FWI hot path -- TEST INFRASTRUCTURE, NOT PRODUCT CODE.

Thin ctypes loader around ``gprfwi_oracle.c`` (plain C99, compiled twice: real and complex for
complex-step derivatives).  Only ``tests/``, ``__graft_entry__.smoke()`` and ``bench.py``'s
``cpu_baseline`` / ``--impl reference`` legs may import this package; the CUDA path
(``paper_2506_20513_b200``) never does, and this package never imports it.

What each function follows in the paper is cited in ``gprfwi_oracle.c``; the readings taken where the
paper is silent are DESIGN.md section 3.  Pins: ``tests/test_oracle_pins.py``.
"""
from __future__ import annotations

import ctypes
import os
import subprocess
from dataclasses import dataclass

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "gprfwi_oracle.c")
_LIB = os.path.join(_HERE, "libgprfwi_oracle.so")

C0 = 299792458.0
MU0 = 4.0e-7 * np.pi
EPS0 = 1.0 / (MU0 * C0 * C0)


def build(force: bool = False) -> str:
    """Compile the oracle with gcc (real + complex objects into one shared library)."""
    if not force and os.path.exists(_LIB) and os.path.getmtime(_LIB) >= os.path.getmtime(_SRC):
        return _LIB
    flags = ["-O2", "-std=c99", "-fPIC", "-fopenmp", "-fno-fast-math"]
    objs = []
    for tag, extra in (("real", []), ("cplx", ["-DORACLE_COMPLEX"])):
        obj = os.path.join(_HERE, f"gprfwi_oracle_{tag}.o")
        subprocess.check_call(["gcc", *flags, *extra, "-c", _SRC, "-o", obj])
        objs.append(obj)
    tmp = _LIB + f".tmp{os.getpid()}"
    subprocess.check_call(["gcc", "-shared", "-fopenmp", *objs, "-o", tmp, "-lm"])
    os.replace(tmp, _LIB)
    return _LIB


class _Params(ctypes.Structure):
    _fields_ = [
        ("nz", ctypes.c_int32), ("nx", ctypes.c_int32),
        ("dx", ctypes.c_double), ("dt", ctypes.c_double),
        ("nt", ctypes.c_int32),
        ("npml", ctypes.c_int32), ("pml_order", ctypes.c_int32),
        ("pml_sigma_max", ctypes.c_double), ("pml_kappa_max", ctypes.c_double),
        ("pml_alpha_max", ctypes.c_double),
        ("nshots", ctypes.c_int32), ("nrec", ctypes.c_int32),
        ("wavelet_per_shot", ctypes.c_int32),
    ]


@dataclass
class Problem:
    """Everything the scheme needs; arrays are converted to float64 / int32 on use."""
    nz: int
    nx: int
    dx: float
    dt: float
    nt: int
    npml: int
    pml_order: int
    pml_sigma_max: float
    pml_kappa_max: float
    pml_alpha_max: float
    src_zx: np.ndarray      # [S][2] full-grid (z, x) cell indices
    rec_zx: np.ndarray      # [S][R][2]
    wavelet: np.ndarray     # [nt] or [S][nt]

    @property
    def nshots(self) -> int:
        return int(np.asarray(self.src_zx).shape[0])

    @property
    def nrec(self) -> int:
        return int(np.asarray(self.rec_zx).shape[1])


_lib = None


def _load():
    global _lib
    if _lib is None:
        _lib = ctypes.CDLL(build())
        _lib.oracle_forward.restype = ctypes.c_int
        _lib.oraclez_forward.restype = ctypes.c_int
        _lib.oracle_gradient.restype = ctypes.c_int
        _lib.oracle_num_threads.restype = ctypes.c_int
    return _lib


def _ptr(a):
    return a.ctypes.data_as(ctypes.c_void_p) if a is not None else None


def _pack(pb: Problem):
    src = np.ascontiguousarray(pb.src_zx, dtype=np.int32).reshape(-1, 2)
    rec = np.ascontiguousarray(pb.rec_zx, dtype=np.int32).reshape(src.shape[0], -1, 2)
    wav = np.ascontiguousarray(pb.wavelet, dtype=np.float64)
    per_shot = 1 if wav.ndim == 2 else 0
    if per_shot:
        assert wav.shape == (src.shape[0], pb.nt)
    else:
        assert wav.shape == (pb.nt,)
    p = _Params(pb.nz, pb.nx, pb.dx, pb.dt, pb.nt, pb.npml, pb.pml_order, pb.pml_sigma_max,
                pb.pml_kappa_max, pb.pml_alpha_max, src.shape[0], rec.shape[1], per_shot)
    return p, src, rec, wav


def num_threads() -> int:
    return int(_load().oracle_num_threads())


def coefficients(eps_r, sigma, dt):
    """Ca, Cb of PAPER.md:291-306 (uE0, uE4).  Complex input gives the complex build."""
    lib = _load()
    cplx = np.iscomplexobj(eps_r) or np.iscomplexobj(sigma)
    dtype = np.complex128 if cplx else np.float64
    e = np.ascontiguousarray(eps_r, dtype=dtype)
    s = np.ascontiguousarray(sigma, dtype=dtype)
    ca = np.empty_like(e)
    cb = np.empty_like(e)
    fn = lib.oraclez_coefficients if cplx else lib.oracle_coefficients
    fn(ctypes.c_int64(e.size), _ptr(e), _ptr(s), ctypes.c_double(dt), _ptr(ca), _ptr(cb))
    return ca, cb


def cpml_profile(n, npml, order, sigma_max, kappa_max, alpha_max, dt, half):
    """(b, c, 1/kappa) 1-D CPML tables; half=0 E-located (n entries), half=1 H-located (n-1)."""
    lib = _load()
    ln = n - 1 if half else n
    b = np.empty(ln)
    c = np.empty(ln)
    ik = np.empty(ln)
    lib.oracle_cpml_profile(ctypes.c_int(n), ctypes.c_int(npml), ctypes.c_int(order),
                            ctypes.c_double(sigma_max), ctypes.c_double(kappa_max),
                            ctypes.c_double(alpha_max), ctypes.c_double(dt), ctypes.c_int(half),
                            _ptr(b), _ptr(c), _ptr(ik))
    return b, c, ik


def _mu(pb, mu_r):
    if mu_r is None:
        return None
    m = np.ascontiguousarray(mu_r, dtype=np.float64)
    assert m.shape == (pb.nz, pb.nx)
    return m


def forward(pb: Problem, eps_r, sigma, want_ez_hist=False, want_h_hist=False, mu_r=None):
    """Algorithm 1.  Returns dict(traces[S][nt][R], ez_hist?, hx_hist?, hy_hist?).
    mu_r: optional [nz][nx] relative permeability (Table 1 `miu`; None = 1)."""
    lib = _load()
    p, src, rec, wav = _pack(pb)
    cplx = np.iscomplexobj(eps_r) or np.iscomplexobj(sigma)
    dtype = np.complex128 if cplx else np.float64
    e = np.ascontiguousarray(eps_r, dtype=dtype)
    s = np.ascontiguousarray(sigma, dtype=dtype)
    assert e.shape == (pb.nz, pb.nx) and s.shape == (pb.nz, pb.nx)
    S, R, nt = p.nshots, p.nrec, pb.nt
    out = {"traces": np.zeros((S, nt, R), dtype=dtype)}
    ez = hx = hy = None
    if want_ez_hist or want_h_hist:
        ez = np.zeros((S, nt + 1, pb.nz, pb.nx), dtype=dtype)
        out["ez_hist"] = ez
    if want_h_hist:
        hx = np.zeros((S, nt + 1, pb.nz - 1, pb.nx), dtype=dtype)
        hy = np.zeros((S, nt + 1, pb.nz, pb.nx - 1), dtype=dtype)
        out["hx_hist"], out["hy_hist"] = hx, hy
    fn = lib.oraclez_forward if cplx else lib.oracle_forward
    mu = _mu(pb, mu_r)
    rc = fn(ctypes.byref(p), _ptr(e), _ptr(s), _ptr(wav), _ptr(src), _ptr(rec),
            _ptr(out["traces"]), _ptr(ez), _ptr(hx), _ptr(hy), _ptr(mu))
    if rc != 0:
        raise ValueError(f"oracle forward failed: code {rc}")
    return out


def gradient(pb: Problem, eps_r, sigma, residual, checkpoint_stride=0, want_traces=False, mu_r=None):
    """Algorithm 2 + chain rule: (grad_eps_r, grad_sigma[, traces]) of sum(residual * traces)."""
    lib = _load()
    p, src, rec, wav = _pack(pb)
    e = np.ascontiguousarray(eps_r, dtype=np.float64)
    s = np.ascontiguousarray(sigma, dtype=np.float64)
    assert e.shape == (pb.nz, pb.nx) and s.shape == (pb.nz, pb.nx)
    res = np.ascontiguousarray(residual, dtype=np.float64)
    assert res.shape == (p.nshots, pb.nt, p.nrec)
    ge = np.zeros_like(e)
    gs = np.zeros_like(e)
    tr = np.zeros((p.nshots, pb.nt, p.nrec)) if want_traces else None
    mu = _mu(pb, mu_r)
    rc = lib.oracle_gradient(ctypes.byref(p), _ptr(e), _ptr(s), _ptr(wav), _ptr(src), _ptr(rec),
                             _ptr(res), ctypes.c_int(checkpoint_stride), _ptr(tr), _ptr(ge), _ptr(gs), _ptr(mu))
    if rc != 0:
        raise ValueError(f"oracle gradient failed: code {rc}")
    return (ge, gs, tr) if want_traces else (ge, gs)
