"""Python binding with the same names as the C-ABI calls (include/gprfwi.h).

Argument marshalling only: tensors must already be fp32, contiguous and on a CUDA device (host
entry points take NumPy arrays); nothing is computed here.
"""
from __future__ import annotations

import ctypes
from dataclasses import dataclass

import numpy as np
import torch

from . import _lib
from ._lib import Params, Plan, UpdateParams, check


def make_params(*, nz, nx, dx, dt, nt, npml, pml_order, pml_sigma_max, pml_kappa_max, pml_alpha_max,
                nshots, nrec, pitch=None, wavelet_per_shot=0, checkpoint_stride=0) -> Params:
    return Params(int(nz), int(nx), int(nx if pitch is None else pitch), float(dx), float(dt), int(nt),
                  int(npml), int(pml_order), float(pml_sigma_max), float(pml_kappa_max),
                  float(pml_alpha_max), int(nshots), int(nrec), int(wavelet_per_shot),
                  int(checkpoint_stride))


def _dev(t: torch.Tensor, name: str, n: int | None = None) -> int:
    if not isinstance(t, torch.Tensor) or not t.is_cuda:
        raise TypeError(f"{name} must be a CUDA tensor (no CPU fallback)")
    if t.dtype != torch.float32 or not t.is_contiguous():
        raise TypeError(f"{name} must be contiguous float32")
    if n is not None and t.numel() < n:
        raise ValueError(f"{name} has {t.numel()} elements, needs {n}")
    return t.data_ptr()


def _plane(t: torch.Tensor, name: str) -> int:
    """A 2-D fp32 CUDA plane whose rows are contiguous (the row stride is passed on as the pitch)."""
    if not isinstance(t, torch.Tensor) or not t.is_cuda or t.dtype != torch.float32 or t.dim() != 2 or t.stride(1) != 1:
        raise TypeError(f"{name} must be a 2-D float32 CUDA tensor with contiguous rows")
    return t.data_ptr()


def _i32(a, shape, name):
    a = np.ascontiguousarray(a, dtype=np.int32)
    if a.shape != shape:
        raise ValueError(f"{name} must have shape {shape}, got {a.shape}")
    return a


def _stream_ptr(stream):
    if stream is None:
        stream = torch.cuda.current_stream()
    return ctypes.c_void_p(stream.cuda_stream)


def gprfwi_workspace_bytes(p: Params, budget_bytes: int = 0):
    """-> (bytes, plan dict); bytes == 0 if the params are invalid or nothing fits the budget."""
    plan = Plan()
    n = _lib.load().gprfwi_workspace_bytes(ctypes.byref(p), int(budget_bytes), ctypes.byref(plan))
    return int(n), plan.as_dict()


def gprfwi_workspace_bytes_host(p: Params, budget_bytes: int = 0) -> int:
    return int(_lib.load().gprfwi_workspace_bytes_host(ctypes.byref(p), int(budget_bytes)))


def split_batch(p: Params, budget_bytes: int = 0, min_shots_per_pass: int = 3):
    """How many equal calls to split p.nshots shots into so that the library's memory plan is a good one
    (host-side planning only, gprfwi_workspace_bytes per candidate): the fewest calls whose plan keeps
    the full history or sends at least `min_shots_per_pass` shots down each adjoint pass (single-shot
    passes leave the launch lanes empty); failing that, the fewest calls that fit at all.
    -> (ncalls, shots per call, plan dict).  Gradients of the calls add; traces concatenate."""
    S = int(p.nshots)
    first = None
    try:
        for ncalls in range(1, S + 1):
            if S % ncalls:
                continue
            p.nshots = S // ncalls
            nbytes, plan = gprfwi_workspace_bytes(p, budget_bytes)
            if nbytes == 0:
                continue
            if first is None:
                first = (ncalls, p.nshots, plan)
            if plan["full_history"] or plan["shots_per_pass"] >= min(min_shots_per_pass, p.nshots):
                return ncalls, p.nshots, plan
    finally:
        p.nshots = S
    if first is None:
        raise ValueError("invalid parameters, or the problem does not fit the budget even one shot at a time")
    return first


def gprfwi_forward(p: Params, eps_r, sigma, wavelet, src_zx, rec_zx, workspace, traces, handle=None,
                   stream=None, mu_r=None):
    """Enqueue Algorithm 1 on `stream`; returns the (new or reused) handle (an int).
    mu_r: optional relative-permeability model (gprfwi_forward_mu; None = 1 everywhere)."""
    lib = _lib.load()
    src = _i32(src_zx, (p.nshots, 2), "src_zx")
    rec = _i32(np.asarray(rec_zx).reshape(p.nshots, p.nrec, 2), (p.nshots, p.nrec, 2), "rec_zx")
    if not (isinstance(workspace, torch.Tensor) and workspace.is_cuda and workspace.dtype == torch.uint8):
        raise TypeError("workspace must be a CUDA uint8 tensor")
    h = ctypes.c_void_p(handle)
    nw = (p.nshots if p.wavelet_per_shot else 1) * p.nt
    code = lib.gprfwi_forward_mu(
        ctypes.byref(h), ctypes.byref(p), _dev(eps_r, "eps_r", p.nz * p.pitch), _dev(sigma, "sigma", p.nz * p.pitch),
        None if mu_r is None else _dev(mu_r, "mu_r", p.nz * p.pitch),
        _dev(wavelet, "wavelet", nw), src.ctypes.data, rec.ctypes.data, workspace.data_ptr(),
        workspace.numel(), _dev(traces, "traces", p.nshots * p.nt * p.nrec) if p.nrec else None,
        _stream_ptr(stream))
    check(code)
    return h.value


def gprfwi_adjoint(handle, p: Params, residual, grad_eps_r, grad_sigma, stream=None):
    """Enqueue Algorithm 2 + chain rule on `stream`."""
    check(_lib.load().gprfwi_adjoint(
        ctypes.c_void_p(handle), _dev(residual, "residual", p.nshots * p.nt * p.nrec) if p.nrec else None,
        _dev(grad_eps_r, "grad_eps_r", p.nz * p.pitch), _dev(grad_sigma, "grad_sigma", p.nz * p.pitch),
        _stream_ptr(stream)))


def gprfwi_residual(d_syn, d_obs, residual, misfit=None, stream=None):
    n = d_syn.numel()
    mp = None
    if misfit is not None:
        if not (misfit.is_cuda and misfit.dtype == torch.float64):
            raise TypeError("misfit must be a CUDA float64 tensor")
        mp = misfit.data_ptr()
    check(_lib.load().gprfwi_residual(_dev(d_syn, "d_syn"), _dev(d_obs, "d_obs", n), _dev(residual, "residual", n),
                                      n, mp, _stream_ptr(stream)))


def gprfwi_gradient_host(p: Params, eps_r, sigma, wavelet, src_zx, rec_zx, d_obs, workspace, traces=None,
                         stream=None):
    """Host-buffer gradient evaluation (NumPy in, NumPy out); copies are inside the call.
    Returns (grad_eps_r, grad_sigma, misfit); `traces` (NumPy, optional) is filled in place."""
    lib = _lib.load()

    def f32(a, n, name):
        a = np.ascontiguousarray(a, dtype=np.float32)
        if a.size < n:
            raise ValueError(f"{name} too small")
        return a

    src = _i32(src_zx, (p.nshots, 2), "src_zx")
    rec = _i32(np.asarray(rec_zx).reshape(p.nshots, p.nrec, 2), (p.nshots, p.nrec, 2), "rec_zx")
    e, s = f32(eps_r, p.nz * p.pitch, "eps_r"), f32(sigma, p.nz * p.pitch, "sigma")
    w = f32(wavelet, (p.nshots if p.wavelet_per_shot else 1) * p.nt, "wavelet")
    d = f32(d_obs, p.nshots * p.nt * p.nrec, "d_obs")
    ge = np.empty((p.nz, p.pitch), dtype=np.float32)
    gs = np.empty((p.nz, p.pitch), dtype=np.float32)
    if traces is not None and not (traces.dtype == np.float32 and traces.flags.c_contiguous):
        raise TypeError("traces must be C-contiguous float32")
    mf = ctypes.c_double(0.0)
    check(lib.gprfwi_gradient_host(
        ctypes.byref(p), e.ctypes.data, s.ctypes.data, w.ctypes.data, src.ctypes.data, rec.ctypes.data,
        d.ctypes.data, workspace.data_ptr(), workspace.numel(),
        traces.ctypes.data if traces is not None else None, ge.ctypes.data, gs.ctypes.data,
        ctypes.byref(mf), _stream_ptr(stream)))
    return ge, gs, mf.value


def make_update_params(*, step, lr_eps_r, lr_sigma, beta1=0.9, beta2=0.999, adam_eps=1e-8, tv_iters=10,
                       tv_rho=1.0, tv_lambda=0.01, tv_alpha=1.0, mask_rows=0, eps_r_min=1.0,
                       sigma_min=0.0) -> UpdateParams:
    return UpdateParams(int(step), float(lr_eps_r), float(lr_sigma), float(beta1), float(beta2), float(adam_eps),
                        int(tv_iters), float(tv_rho), float(tv_lambda), float(tv_alpha), int(mask_rows),
                        float(eps_r_min), float(sigma_min))


def gprfwi_update_workspace_bytes(nz: int, pitch: int) -> int:
    return int(_lib.load().gprfwi_update_workspace_bytes(int(nz), int(pitch)))


def gprfwi_update(nz, nx, pitch, u: UpdateParams, eps_r, sigma, grad_eps_r, grad_sigma, m_eps_r, v_eps_r,
                  m_sigma, v_sigma, workspace, stream=None):
    """Enqueue one optimiser step (TV term, mask, Adam, clamps) on `stream`; all planes updated in place."""
    n = nz * pitch
    ptrs = [_dev(t, nm, n) for t, nm in ((eps_r, "eps_r"), (sigma, "sigma"), (grad_eps_r, "grad_eps_r"),
                                          (grad_sigma, "grad_sigma"), (m_eps_r, "m_eps_r"), (v_eps_r, "v_eps_r"),
                                          (m_sigma, "m_sigma"), (v_sigma, "v_sigma"))]
    if not (isinstance(workspace, torch.Tensor) and workspace.is_cuda and workspace.dtype == torch.uint8):
        raise TypeError("workspace must be a CUDA uint8 tensor")
    check(_lib.load().gprfwi_update(int(nz), int(nx), int(pitch), ctypes.byref(u), *ptrs, workspace.data_ptr(),
                                    workspace.numel(), _stream_ptr(stream)))


def gprfwi_update_noalloc(nz, nx, pitch, u: UpdateParams, eps_r, sigma, grad_eps_r, grad_sigma, m_eps_r, v_eps_r,
                          m_sigma, v_sigma, stream=None):
    """gprfwi_update with the TV scratch in the library's fixed device array: no workspace, no allocation.
    Raises GprfwiError(ETOOBIG) beyond gprfwi_update_noalloc_max_bytes(); overlapping calls race (see the header)."""
    n = nz * pitch
    ptrs = [_dev(t, nm, n) for t, nm in ((eps_r, "eps_r"), (sigma, "sigma"), (grad_eps_r, "grad_eps_r"),
                                          (grad_sigma, "grad_sigma"), (m_eps_r, "m_eps_r"), (v_eps_r, "v_eps_r"),
                                          (m_sigma, "m_sigma"), (v_sigma, "v_sigma"))]
    check(_lib.load().gprfwi_update_noalloc(int(nz), int(nx), int(pitch), ctypes.byref(u), *ptrs, _stream_ptr(stream)))


def gprfwi_update_noalloc_max_bytes() -> int:
    return int(_lib.load().gprfwi_update_noalloc_max_bytes())


def gprfwi_lowpass(x: torch.Tensor, out: torch.Tensor, taps: torch.Tensor, stream=None):
    """Zero-phase FIR along time of x[nseries][nt][nrec] (or [nseries][nt]) into `out` (multiscale stages)."""
    if x.dim() == 2:
        nseries, nt, nrec = x.shape[0], x.shape[1], 1
    else:
        nseries, nt, nrec = x.shape
    check(_lib.load().gprfwi_lowpass(_dev(x, "x"), _dev(out, "out", x.numel()), int(nseries), int(nt), int(nrec),
                                     _dev(taps, "taps"), int(taps.numel()), _stream_ptr(stream)))
    return out


def gprfwi_lowpass_design(dt: float, f_cut: float, ntaps: int = 0) -> np.ndarray:
    """Taps of the stage filter (host call into the library; reading R21) as a float32 NumPy array."""
    lib = _lib.load()
    n = int(lib.gprfwi_lowpass_design(float(dt), float(f_cut), int(ntaps), None))
    check(min(n, 0))
    taps = np.empty(n, dtype=np.float32)
    check(min(int(lib.gprfwi_lowpass_design(float(dt), float(f_cut), n, taps.ctypes.data)), 0))
    return taps


def gprfwi_restrict(fine: torch.Tensor, coarse: torch.Tensor = None, stream=None) -> torch.Tensor:
    """Full-weighting 2:1 restriction of a model plane [nz][nx] -> [(nz+1)//2][(nx+1)//2] (reading R23)."""
    nz, nx = fine.shape
    if coarse is None:
        coarse = torch.empty(((nz + 1) // 2, (nx + 1) // 2), dtype=torch.float32, device=fine.device)
    check(_lib.load().gprfwi_restrict(_plane(fine, "fine"), nz, nx, fine.stride(0), _plane(coarse, "coarse"),
                                      coarse.stride(0), _stream_ptr(stream)))
    return coarse


def gprfwi_prolong_add(coarse: torch.Tensor, fine: torch.Tensor, scale: float = 1.0, stream=None) -> torch.Tensor:
    """fine += scale * bilinear prolongation of coarse (reading R23)."""
    nz, nx = fine.shape
    if tuple(coarse.shape) != ((nz + 1) // 2, (nx + 1) // 2):
        raise ValueError("coarse must have shape ((nz+1)//2, (nx+1)//2)")
    check(_lib.load().gprfwi_prolong_add(_plane(coarse, "coarse"), coarse.stride(0), float(scale), _plane(fine, "fine"),
                                         nz, nx, fine.stride(0), _stream_ptr(stream)))
    return fine


class Simulation:
    """Owns the device buffers (torch) and the library handle for one problem."""

    def __init__(self, p: Params, src_zx, rec_zx, wavelet, device="cuda:0", budget_bytes: int = 0):
        self.p = p
        self.device = torch.device(device)
        self.src_zx, self.rec_zx = src_zx, rec_zx
        nbytes, self.plan = gprfwi_workspace_bytes(p, budget_bytes)
        if nbytes == 0:
            raise ValueError("invalid parameters or nothing fits the memory budget")
        self.workspace = torch.empty(nbytes, dtype=torch.uint8, device=self.device)
        self.wavelet = torch.as_tensor(np.ascontiguousarray(wavelet, dtype=np.float32), device=self.device)
        self.traces = torch.empty((p.nshots, p.nt, p.nrec), dtype=torch.float32, device=self.device)
        self.grad_eps_r = torch.empty((p.nz, p.pitch), dtype=torch.float32, device=self.device)
        self.grad_sigma = torch.empty((p.nz, p.pitch), dtype=torch.float32, device=self.device)
        self.handle = None
        self._models = None

    def forward(self, eps_r: torch.Tensor, sigma: torch.Tensor, stream=None, mu_r=None) -> torch.Tensor:
        self._models = (eps_r, sigma, mu_r)  # must stay alive and unmodified until the adjoint
        self.handle = gprfwi_forward(self.p, eps_r, sigma, self.wavelet, self.src_zx, self.rec_zx,
                                     self.workspace, self.traces, self.handle, stream, mu_r)
        return self.traces

    def adjoint(self, residual: torch.Tensor, stream=None):
        gprfwi_adjoint(self.handle, self.p, residual, self.grad_eps_r, self.grad_sigma, stream)
        return self.grad_eps_r, self.grad_sigma

    def launch_count(self) -> int:
        return int(_lib.load().gprfwi_launch_count(ctypes.c_void_p(self.handle)))

    def close(self):
        if self.handle is not None:
            _lib.load().gprfwi_release(ctypes.c_void_p(self.handle))
            self.handle = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass


def invert(sim: "Simulation", eps_r: torch.Tensor, sigma: torch.Tensor, d_obs: torch.Tensor, *, iterations: int,
           lr_eps_r: float, lr_sigma: float, mask_rows: int = 0, tv_iters: int = 10, tv_lambda: float = 0.01,
           tv_alpha: float = 1.0, eps_r_min: float = 1.0, sigma_min: float = 0.0, callback=None):
    """The paper's inversion loop as a sequence of C-ABI calls, nothing computed here:
    per iteration gprfwi_forward -> gprfwi_residual (+ misfit) -> gprfwi_adjoint -> gprfwi_update
    (TV term, source mask, Adam with one learning rate per parameter, clamps).  `eps_r` and `sigma`
    are updated in place; returns the list of misfits 0.5*||d_syn - d_obs||^2 (one per iteration,
    evaluated BEFORE that iteration's update)."""
    p = sim.p
    if p.pitch != p.nx:
        raise ValueError("invert() expects unpadded models (pitch == nx)")
    dev = sim.device
    res = torch.empty_like(d_obs)
    misfit = torch.zeros(1, dtype=torch.float64, device=dev)
    state = [torch.zeros_like(eps_r) for _ in range(4)]
    ws = torch.empty(gprfwi_update_workspace_bytes(p.nz, p.pitch), dtype=torch.uint8, device=dev)
    history = []
    for it in range(1, iterations + 1):
        traces = sim.forward(eps_r, sigma)
        misfit.zero_()
        gprfwi_residual(traces, d_obs, res, misfit)
        ge, gs = sim.adjoint(res)
        u = make_update_params(step=it, lr_eps_r=lr_eps_r, lr_sigma=lr_sigma, tv_iters=tv_iters,
                               tv_lambda=tv_lambda, tv_alpha=tv_alpha, mask_rows=mask_rows,
                               eps_r_min=eps_r_min, sigma_min=sigma_min)
        gprfwi_update(p.nz, p.nx, p.pitch, u, eps_r, sigma, ge, gs, state[0], state[1], state[2], state[3], ws)
        history.append(float(misfit.item()))
        if callback is not None:
            callback(it, history[-1])
    return history


@dataclass
class Stage:
    """One stage of a staged inversion: the two-stage learning-rate strategy of PAPER.md:547 (eps_r first,
    then both: set lr_sigma = 0 in the first stage) and / or one band of the multiscale strategy of
    PAPER.md:529-531 (`f_cut` = low-pass corner in Hz applied to the wavelet and the observed data;
    None = full band)."""
    iterations: int
    lr_eps_r: float
    lr_sigma: float
    f_cut: float | None = None
    ntaps: int = 0
    coarsen: bool = False      # run this stage on the 2:1 coarse grid (reading R23)


def coarse_problem(p: Params, src_zx, rec_zx):
    """The 2:1 coarse counterpart of a problem (reading R23): same dt and nt, dx doubled, CPML thickness halved
    (rounded up) with sigma_max halved (it scales like 1/dx), sources and receivers on the nearest coarse node
    inside the PEC ring.  Host-side bookkeeping only."""
    nzc, nxc = (p.nz + 1) // 2, (p.nx + 1) // 2
    pc = make_params(nz=nzc, nx=nxc, dx=2.0 * p.dx, dt=p.dt, nt=p.nt, npml=(p.npml + 1) // 2, pml_order=p.pml_order,
                     pml_sigma_max=0.5 * p.pml_sigma_max, pml_kappa_max=p.pml_kappa_max,
                     pml_alpha_max=p.pml_alpha_max, nshots=p.nshots, nrec=p.nrec,
                     wavelet_per_shot=p.wavelet_per_shot)

    def coarse_idx(a):
        a = (np.asarray(a, dtype=np.int64) + 1) // 2
        a[..., 0] = np.clip(a[..., 0], 1, nzc - 2)
        a[..., 1] = np.clip(a[..., 1], 1, nxc - 2)
        return a.astype(np.int32)

    return pc, coarse_idx(src_zx), coarse_idx(np.asarray(rec_zx).reshape(p.nshots, p.nrec, 2))


def _invert_coarse(sim, eps_r, sigma, d_obs, wavelet, st, cb, update_kw):
    """One stage on the coarse grid: restrict the models, invert there, prolong the model UPDATES back."""
    pc, src_c, rec_c = coarse_problem(sim.p, sim.src_zx, sim.rec_zx)
    simc = Simulation(pc, src_c, rec_c, np.zeros(wavelet.numel(), dtype=np.float32), sim.device)
    simc.wavelet = wavelet
    try:
        e0, s0 = gprfwi_restrict(eps_r), gprfwi_restrict(sigma)
        ec, sc = e0.clone(), s0.clone()
        kw = dict(update_kw)
        if "mask_rows" in kw:
            kw["mask_rows"] = (kw["mask_rows"] + 1) // 2
        hist = invert(simc, ec, sc, d_obs, iterations=st.iterations, lr_eps_r=st.lr_eps_r, lr_sigma=st.lr_sigma,
                      callback=cb, **kw)
        gprfwi_prolong_add(ec.sub_(e0), eps_r)
        gprfwi_prolong_add(sc.sub_(s0), sigma)
        eps_r.clamp_(min=kw.get("eps_r_min", 1.0))
        sigma.clamp_(min=kw.get("sigma_min", 0.0))
    finally:
        simc.close()
    return hist


def invert_staged(sim: "Simulation", eps_r: torch.Tensor, sigma: torch.Tensor, d_obs: torch.Tensor, stages,
                  callback=None, **update_kw):
    """Stage driver (reading R21): per stage, low-pass the source wavelet and
    d_obs with gprfwi_lowpass when the stage has a corner frequency, then run invert() with the stage's
    learning rates.  Adam's moments and step counter restart at every stage; a parameter whose learning
    rate is 0 does not move.  Returns one misfit list per stage; `callback(stage, iteration, misfit)`."""
    full = sim.wavelet
    dev = sim.device
    out = []
    try:
        for k, st in enumerate(stages):
            w, d = full, d_obs
            if st.f_cut is not None:
                taps = torch.as_tensor(gprfwi_lowpass_design(sim.p.dt, st.f_cut, st.ntaps), device=dev)
                w2 = full.reshape(-1, sim.p.nt)
                w = gprfwi_lowpass(w2, torch.empty_like(w2), taps).reshape(full.shape)
                d = gprfwi_lowpass(d_obs, torch.empty_like(d_obs), taps)
            sim.wavelet = w
            cb = None if callback is None else (lambda it, mf, k=k: callback(k, it, mf))
            if st.coarsen:
                out.append(_invert_coarse(sim, eps_r, sigma, d, w, st, cb, update_kw))
                continue
            out.append(invert(sim, eps_r, sigma, d, iterations=st.iterations, lr_eps_r=st.lr_eps_r,
                              lr_sigma=st.lr_sigma, callback=cb, **update_kw))
    finally:
        sim.wavelet = full
    return out
