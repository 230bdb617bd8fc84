"""Seeded synthetic inputs for the GPR-FWI hot path (BASELINE.json configs 1-5).

This module serves BOTH the float64 oracle (``oracle/``) and the CUDA path
(``paper_2506_20513_b200``).  It holds none of the method's arithmetic: it only makes models
(eps_r, sigma), acquisition geometry, the source wavelet and the *scalar* CPML parameters that the
method takes as inputs.  Everything is a pure function of (config, seed); nothing is read from disk
and nothing comes from either implementation.  Recipes: DESIGN.md section 5 (after SURVEY.md
section 8(d)); they stand in for the paper's own models (landfill, Overthrust, field data), which
are not available.

All model arrays are float32 (what the GPU consumes); the oracle up-casts the same values.
"""
from __future__ import annotations

from dataclasses import dataclass, field, replace

import numpy as np

C0 = 299792458.0
MU0 = 4.0e-7 * np.pi
EPS0 = 1.0 / (MU0 * C0 * C0)
ETA0 = float(np.sqrt(MU0 / EPS0))

BASE_SEED = 20250620


@dataclass
class Workload:
    name: str
    nz: int                 # full grid incl. CPML
    nx: int
    dx: float
    dt: float
    nt: int
    npml: int
    pml_order: int
    pml_sigma_max: float
    pml_kappa_max: float
    pml_alpha_max: float
    freq: float
    eps_r: np.ndarray       # [nz][nx] float32, model the gradient is taken at
    sigma: np.ndarray
    eps_r_obs: np.ndarray | None    # model that generates d_obs (None: residual is random)
    sigma_obs: np.ndarray | None
    wavelet: np.ndarray     # [nt] float32, line current (A) during step n, sampled at (n+1/2)dt
    src_zx: np.ndarray      # [S][2] int32
    rec_zx: np.ndarray      # [S][R][2] int32
    seed: int = BASE_SEED
    notes: dict = field(default_factory=dict)

    @property
    def nshots(self) -> int:
        return int(self.src_zx.shape[0])

    @property
    def nrec(self) -> int:
        return int(self.rec_zx.shape[1])

    @property
    def cell_updates(self) -> int:
        """forward + adjoint work: 2 * NZ * NX * nt * S."""
        return 2 * self.nz * self.nx * self.nt * self.nshots

    def subset(self, shots, nt: int | None = None) -> "Workload":
        """Same problem restricted to some shots (and optionally fewer time steps)."""
        shots = np.asarray(shots, dtype=np.int64)
        nt = self.nt if nt is None else int(nt)
        return replace(self, name=f"{self.name}[shots={shots.tolist()},nt={nt}]", nt=nt,
                       wavelet=self.wavelet[:nt].copy(), src_zx=self.src_zx[shots].copy(),
                       rec_zx=self.rec_zx[shots].copy())


# ------------------------------------------------------------------------------------------------
# ingredients
# ------------------------------------------------------------------------------------------------
def ricker(nt: int, dt: float, freq: float, amp: float = 1.0) -> np.ndarray:
    """Ricker current sampled at (n + 1/2) dt, delayed by sqrt(2)/f (reading R9)."""
    t = (np.arange(nt, dtype=np.float64) + 0.5) * dt
    tau = t - np.sqrt(2.0) / freq
    z = (np.pi * freq) ** 2 * tau * tau
    return (amp * (1.0 - 2.0 * z) * np.exp(-z)).astype(np.float32)


def cpml_defaults(dx: float, freq: float, eps_ref: float, order: int = 3):
    """Scalar CPML parameters handed to both implementations (reading R4)."""
    sigma_max = 0.8 * (order + 1) / (ETA0 * dx * np.sqrt(eps_ref))
    kappa_max = 1.0
    alpha_max = 0.1 * 2.0 * np.pi * EPS0 * freq
    return order, float(sigma_max), float(kappa_max), float(alpha_max)


def pad_edge(interior: np.ndarray, npml: int) -> np.ndarray:
    """Edge-replicate an interior model into the CPML (reading R10)."""
    return np.pad(interior, npml, mode="edge").astype(np.float32)


def line_geometry(nz_int: int, nx_int: int, npml: int, nshots: int, nrec: int, depth_cells: int = 5,
                  per_shot_receivers: bool = False):
    """Sources and receivers on the row iz = npml + depth_cells, evenly spaced in x."""
    iz = npml + depth_cells
    sx = npml + np.floor((np.arange(nshots) + 0.5) * nx_int / nshots).astype(np.int64)
    rx = npml + np.floor((np.arange(nrec) + 0.5) * nx_int / nrec).astype(np.int64)
    src = np.stack([np.full(nshots, iz), sx], axis=1).astype(np.int32)
    rec1 = np.stack([np.full(nrec, iz), rx], axis=1).astype(np.int32)
    rec = np.broadcast_to(rec1, (nshots, nrec, 2)).copy()
    return src, rec


def acquisition(src0_zx, src_step_zx, steps: int, rec0_zx, rec_step_zx, nrx: int,
                fixed_receiver: bool = False):
    """Acquisition of PAPER.md:184-199 (Table 1: source_location, source_step, step, receiver_location,
    receiver_step, nrx, Fixedreceiver) in grid cells.  Shot k fires at src0 + k*src_step; its receivers
    sit at rec0 + j*rec_step (j < nrx), shifted by k*src_step as well unless `fixed_receiver`
    (a moving source-receiver array; nrx = 1 gives a common-offset profile)."""
    k = np.arange(steps, dtype=np.int64)[:, None]
    j = np.arange(nrx, dtype=np.int64)[:, None]
    src = np.asarray(src0_zx, dtype=np.int64)[None, :] + k * np.asarray(src_step_zx, dtype=np.int64)[None, :]
    rec1 = np.asarray(rec0_zx, dtype=np.int64)[None, :] + j * np.asarray(rec_step_zx, dtype=np.int64)[None, :]
    rec = np.broadcast_to(rec1, (steps, nrx, 2)).copy()
    if not fixed_receiver:
        rec += (src - src[:1])[:, None, :]
    return src.astype(np.int32), rec.astype(np.int32)


def with_geometry(wl: "Workload", src_zx, rec_zx, name: str | None = None) -> "Workload":
    """Same models and wavelet, other acquisition (positions must lie inside the PEC ring)."""
    src = np.ascontiguousarray(src_zx, dtype=np.int32)
    rec = np.ascontiguousarray(rec_zx, dtype=np.int32)
    assert src.ndim == 2 and rec.ndim == 3 and rec.shape[0] == src.shape[0]
    for a, n in ((src[:, 0], wl.nz), (src[:, 1], wl.nx), (rec[..., 0], wl.nz), (rec[..., 1], wl.nx)):
        assert a.min() >= 1 and a.max() <= n - 2, "position on or outside the PEC ring"
    return replace(wl, name=name or wl.name + "+geometry", src_zx=src, rec_zx=rec)


def _gauss2d(nz, nx, cz, cx, std):
    z = np.arange(nz, dtype=np.float64)[:, None]
    x = np.arange(nx, dtype=np.float64)[None, :]
    return np.exp(-((z - cz) ** 2 + (x - cx) ** 2) / (2.0 * std * std))


def _smooth_noise(rng, nz, nx, std, lo, hi):
    """White noise -> separable Gaussian filter (reflect) -> affine map to [lo, hi]."""
    from scipy.ndimage import gaussian_filter
    f = gaussian_filter(rng.standard_normal((nz, nx)), std, mode="reflect")
    f = (f - f.min()) / (f.max() - f.min())
    return lo + (hi - lo) * f


def _finish(name, eps_i, sig_i, eps_obs_i, sig_obs_i, npml, dx, dt, nt, freq, nshots, nrec, seed,
            notes=None, geometry=None):
    nz_int, nx_int = eps_i.shape
    order, smax, kmax, amax = cpml_defaults(dx, freq, float(np.mean(eps_i)))
    if geometry is None:
        geometry = line_geometry(nz_int, nx_int, npml, nshots, nrec)
    src, rec = geometry
    return Workload(
        name=name, nz=nz_int + 2 * npml, nx=nx_int + 2 * npml, dx=dx, dt=dt, nt=nt, npml=npml,
        pml_order=order, pml_sigma_max=smax, pml_kappa_max=kmax, pml_alpha_max=amax, freq=freq,
        eps_r=pad_edge(eps_i, npml), sigma=pad_edge(sig_i, npml),
        eps_r_obs=None if eps_obs_i is None else pad_edge(eps_obs_i, npml),
        sigma_obs=None if sig_obs_i is None else pad_edge(sig_obs_i, npml),
        wavelet=ricker(nt, dt, freq), src_zx=src, rec_zx=rec, seed=seed, notes=notes or {})


# ------------------------------------------------------------------------------------------------
# BASELINE.json configs
# ------------------------------------------------------------------------------------------------
def config1(nt: int = 800) -> Workload:
    """Tiny PR1 ref: 100x100 interior + 10-cell CPML, two layers, one shot, 10 receivers;
    d_obs from the same model plus a disc (eps_r 16, sigma 10 mS/m), integer-cell geometry."""
    n, npml = 100, 10
    j = np.arange(n)[:, None] * np.ones((1, n), dtype=np.int64)
    i = np.ones((n, 1), dtype=np.int64) * np.arange(n)[None, :]
    eps = np.where(j < 50, 4.0, 9.0)
    sig = np.full((n, n), 1.0e-3)
    disc = (i - 50) ** 2 + (j - 70) ** 2 <= 100
    eps_o = np.where(disc, 16.0, eps)
    sig_o = np.where(disc, 1.0e-2, sig)
    return _finish("config1-tiny", eps, sig, eps_o, sig_o, npml, 0.01, 2e-11, nt, 400e6, 1, 10,
                   BASE_SEED + 1, notes={"disc_nodes": int(disc.sum())})


def config2(nshots: int = 20, nrec: int = 100, nt: int = 3000) -> Workload:
    """Paper-scale synthetic: 200x400 interior + 20-cell CPML, 3 layers + Gaussian anomalies."""
    seed = BASE_SEED + 2
    rng = np.random.Generator(np.random.PCG64(seed))
    nz, nx, npml = 200, 400, 20
    j = np.arange(nz)[:, None] * np.ones((1, nx), dtype=np.int64)
    eps = np.where(j < nz // 3, 4.0, np.where(j < 2 * nz // 3, 6.0, 9.0)).astype(np.float64)
    sig = np.where(j < nz // 3, 1e-3, np.where(j < 2 * nz // 3, 3e-3, 5e-3)).astype(np.float64)
    for _ in range(3):
        sign = rng.choice([-1.0, 1.0])
        cz, cx = rng.uniform(0.15 * nz, 0.85 * nz), rng.uniform(0.15 * nx, 0.85 * nx)
        eps = eps + sign * 3.0 * _gauss2d(nz, nx, cz, cx, rng.uniform(8, 25))
    for _ in range(2):
        cz, cx = rng.uniform(0.15 * nz, 0.85 * nz), rng.uniform(0.15 * nx, 0.85 * nx)
        peak = rng.uniform(10e-3, 20e-3)
        sig = sig + peak * _gauss2d(nz, nx, cz, cx, rng.uniform(8, 25))
    eps = np.maximum(eps, 1.0)
    g = _gauss2d(nz, nx, nz / 2, nx / 2, 15.0)
    return _finish("config2-paper-scale", eps, sig, eps + 2.0 * g, sig + 5e-3 * g, npml, 0.01, 2e-11,
                   nt, 400e6, nshots, nrec, seed)


def config3(nshots: int = 60, nrec: int = 200, nt: int = 4000) -> Workload:
    """Larger survey: 500x1000 interior + 20-cell CPML, smooth random fields."""
    seed = BASE_SEED + 3
    rng = np.random.Generator(np.random.PCG64(seed))
    nz, nx, npml = 500, 1000, 20
    eps = _smooth_noise(rng, nz, nx, 10.0, 3.0, 12.0)
    sig = _smooth_noise(rng, nz, nx, 10.0, 0.5e-3, 20e-3)
    eps2 = _smooth_noise(rng, nz, nx, 10.0, 3.0, 12.0)
    sig2 = _smooth_noise(rng, nz, nx, 10.0, 0.5e-3, 20e-3)
    return _finish("config3-larger-survey", eps, sig, 0.9 * eps + 0.1 * eps2, 0.9 * sig + 0.1 * sig2,
                   npml, 0.01, 2e-11, nt, 400e6, nshots, nrec, seed)


def _inclusions(rng, nz, nx, eps, sig):
    z = np.arange(nz)[:, None]
    x = np.arange(nx)[None, :]
    for k in range(20):
        size = int(rng.integers(10, 61))
        cz, cx = int(rng.integers(size, nz - size)), int(rng.integers(size, nx - size))
        e = rng.uniform(4.0, 16.0)
        s = float(np.exp(rng.uniform(np.log(0.1e-3), np.log(30e-3))))
        if k < 10:
            m = (np.abs(z - cz) <= size // 2) & (np.abs(x - cx) <= size // 2)
        else:
            m = (z - cz) ** 2 + (x - cx) ** 2 <= (size // 2) ** 2
        eps = np.where(m, e, eps)
        sig = np.where(m, s, sig)
    return eps, sig


def config4(nshots: int = 100, nrec: int = 400, nt: int = 6000) -> Workload:
    """High-frequency: 1000x2000 interior + 30-cell CPML, 5 layers + 20 inclusions, 1.2 GHz."""
    seed = BASE_SEED + 4
    nz, nx, npml = 1000, 2000, 30
    layer = np.minimum(np.arange(nz) // (nz // 5), 4)[:, None] * np.ones((1, nx), dtype=np.int64)
    eps0 = np.array([4.0, 7.0, 10.0, 13.0, 16.0])[layer]
    sig0 = np.array([0.1e-3, 1e-3, 5e-3, 15e-3, 30e-3])[layer]
    eps, sig = _inclusions(np.random.Generator(np.random.PCG64(seed)), nz, nx, eps0, sig0)
    eps_o, sig_o = _inclusions(np.random.Generator(np.random.PCG64(seed + 1000)), nz, nx, eps0, sig0)
    return _finish("config4-high-frequency", eps, sig, eps_o, sig_o, npml, 0.005, 1e-11, nt, 1.2e9,
                   nshots, nrec, seed)


def crosshole(nt: int = 1000, nrec: int = 200) -> Workload:
    """Shapes of the paper's cross-hole experiment (section 4.1): 120 x 220 cells incl. a
    10-cell CPML, dx = 0.05 m, dt = 1e-10 s, 1e-7 s window, one 100 MHz source in one hole and `nrec`
    receivers down a line 5 m away.  The models are a seeded stand-in (three layers, three anomalies and
    a thin channel with eps_r and sigma placed differently), not the paper's landfill model."""
    seed = BASE_SEED + 6
    npml, nz, nx = 10, 200, 100                      # interior; z is the long (depth) axis
    rng = np.random.Generator(np.random.PCG64(seed))
    layer = np.minimum(np.arange(nz) // 70, 2)[:, None] * np.ones((1, nx), dtype=np.int64)
    eps = np.array([5.0, 8.0, 11.0])[layer]
    sig = np.array([1e-3, 3e-3, 6e-3])[layer]
    eps_o, sig_o = eps.copy(), sig.copy()
    z = np.arange(nz)[:, None]; x = np.arange(nx)[None, :]
    for k in range(3):
        cz, cx, r = int(rng.integers(30, nz - 30)), int(rng.integers(30, nx - 30)), int(rng.integers(6, 12))
        m = (z - cz) ** 2 + (x - cx) ** 2 <= r * r
        eps_o = np.where(m, rng.uniform(3.0, 16.0), eps_o)
        m2 = (z - cz - 8) ** 2 + (x - cx + 5) ** 2 <= r * r          # sigma anomaly displaced
        sig_o = np.where(m2, float(np.exp(rng.uniform(np.log(5e-3), np.log(3e-2)))), sig_o)
    chan = (np.abs(z - (60 + x // 3)) <= 1) & (x > 25) & (x < 80)
    eps_o = np.where(chan, 14.0, eps_o); sig_o = np.where(chan, 2e-2, sig_o)
    src, rec = acquisition((npml + 10, npml + 10), (0, 0), 1, (npml, npml + 89), (1, 0), min(nrec, nz),
                           fixed_receiver=True)
    return _finish("crosshole-4.1-shapes", eps, sig, eps_o, sig_o, npml, 0.05, 1e-10, nt, 100e6, 1, nrec,
                   seed, geometry=(src, rec))


def config5(n: int = 512, batch: int = 1, nt: int = 1000, nrec: int = 64) -> Workload:
    """Stencil sweep: N x N TOTAL cells incl. 20-cell CPML, i.i.d. uniform models, per-shot
    receiver lines.  dx, dt, f are not given by BASELINE.json: 0.01 m, 2e-11 s, 400 MHz."""
    seed = BASE_SEED + 5
    rng = np.random.Generator(np.random.PCG64(seed + n))
    npml = 20
    ni = n - 2 * npml
    eps = rng.uniform(1.0, 20.0, (ni, ni))
    sig = rng.uniform(0.0, 0.05, (ni, ni))
    return _finish(f"config5-sweep-{n}x{n}-b{batch}", eps, sig, None, None, npml, 0.01, 2e-11, nt,
                   400e6, batch, nrec, seed, geometry=line_geometry(ni, ni, npml, batch, nrec))


def random_residual(wl: Workload, trace_rms: float = 1.0, seed: int | None = None) -> np.ndarray:
    """Seeded N(0, trace_rms) residual [S][nt][R] (a valid input for J^T); sample 0 zeroed."""
    rng = np.random.Generator(np.random.PCG64((wl.seed if seed is None else seed) + 7))
    r = rng.standard_normal((wl.nshots, wl.nt, wl.nrec)) * trace_rms
    r[:, 0, :] = 0.0
    return r.astype(np.float32)


def small_random(nz=44, nx=52, nt=120, npml=8, nshots=2, nrec=5, seed=1234, lossy=True,
                 dx=0.01, dt=2e-11, freq=400e6) -> Workload:
    """Tiny heterogeneous lossy problem with scattered interior sources/receivers (tests only)."""
    rng = np.random.Generator(np.random.PCG64(seed))
    eps = rng.uniform(2.0, 9.0, (nz, nx))
    sig = rng.uniform(0.0, 0.02, (nz, nx)) if lossy else np.zeros((nz, nx))
    order, smax, kmax, amax = cpml_defaults(dx, freq, float(eps.mean()))
    lo = npml + 2 if npml > 0 else 2
    src = np.stack([rng.integers(lo, nz - lo, nshots), rng.integers(lo, nx - lo, nshots)], 1)
    rec = np.stack([rng.integers(1, nz - 1, (nshots, nrec)), rng.integers(1, nx - 1, (nshots, nrec))], 2)
    return Workload(name="small-random", nz=nz, nx=nx, dx=dx, dt=dt, nt=nt, npml=npml, pml_order=order,
                    pml_sigma_max=smax, pml_kappa_max=kmax, pml_alpha_max=amax, freq=freq,
                    eps_r=eps.astype(np.float32), sigma=sig.astype(np.float32), eps_r_obs=None,
                    sigma_obs=None, wavelet=ricker(nt, dt, freq), src_zx=src.astype(np.int32),
                    rec_zx=rec.astype(np.int32), seed=seed)
