"""TEST INFRASTRUCTURE, NOT PRODUCT CODE -- float64 NumPy statement of the iteration epilogue
(SURVEY 8(a) row a7): TV term of Algorithm 3 (Eq. (17)), gradient mask near the
sources, Adam step with one learning rate per parameter (Eqs. (14)-(15),
PAPER.md:105-112) and the clamps of PAPER.md:258-260.  Shares nothing with csrc/.

Readings (R18-R20).  The paper lists Algorithm 3's steps without constants or a
definition of `*_tv_grad`; the reading below is the one both sides implement.

Pins (tests/test_oracle_pins.py): Adam's first step equals -lr g/(|g| + eps) (closed form of
Eqs. (14)-(15) at t = 1), masked rows do not move, clamps hold; shrink(v, t) = v max(1 - t/|v|, 0)
(Eq. (17)); a constant X gives tv_grad = 0; the U update solves (I + rho D^T D) U = U0 + rho D^T (Z - B)
in the limit of many sweeps (checked with one dense solve on a tiny grid); run to convergence the
iteration reaches the minimiser of 1/2 |U - U0|^2 + lambda TV(U), checked against its closed form for a
two-level periodic stripe along either axis (plateaus approach by 2 lambda / L, and merge at the mean
for large lambda).  What the paper does not fix -- the constants, the scaling by max|X|, one Jacobi
sweep per iteration, stopping after n_it iterations -- stays a reading (R20): at the default n_it the
TV term is PARITY UNPINNED against the paper, which prints no value to compare with.
"""
import numpy as np


def shrink(vx, vz, t):
    """Isotropic soft threshold, Eq. (17): v * max(1 - t/|v|, 0)."""
    nrm = np.sqrt(vx * vx + vz * vz)
    f = np.where(nrm > t, 1.0 - t / np.where(nrm > t, nrm, 1.0), 0.0)
    return f * vx, f * vz


def tv_gradient(x, iters=10, rho=1.0, lam=0.01, alpha=1.0):
    """Algorithm 3 (reading R20): returns alpha * (X - s U) after `iters` split-variable iterations."""
    x = np.asarray(x, dtype=np.float64)
    s = np.max(np.abs(x))
    u0 = x / s if s > 0 else np.zeros_like(x)
    u = u0.copy()
    zx = np.zeros_like(u); zz = np.zeros_like(u); bx = np.zeros_like(u); bz = np.zeros_like(u)
    for _ in range(iters):
        wx, wz = zx - bx, zz - bz
        div = (np.roll(wx, 1, axis=1) - wx) + (np.roll(wz, 1, axis=0) - wz)          # D^T (Z - B)
        nb = np.roll(u, 1, axis=1) + np.roll(u, -1, axis=1) + np.roll(u, 1, axis=0) + np.roll(u, -1, axis=0)
        u = (u0 + rho * div + rho * nb) / (1.0 + 4.0 * rho)                           # one Jacobi sweep
        gx = np.roll(u, -1, axis=1) - u                                               # D U, circular forward
        gz = np.roll(u, -1, axis=0) - u
        zx, zz = shrink(gx + bx, gz + bz, lam / rho)
        bx = bx + gx - zx
        bz = bz + gz - zz
    return alpha * (x - s * u)


def adam_step(x, g, m, v, step, lr, beta1=0.9, beta2=0.999, eps=1e-8, mask_rows=0, xmin=-np.inf):
    """Eqs. (14)-(15) with the epsilon outside the root (reading R19); returns (x, m, v)."""
    g = np.array(g, dtype=np.float64)
    g[:mask_rows] = 0.0                                                               # reading R18
    m = beta1 * m + (1.0 - beta1) * g
    v = beta2 * v + (1.0 - beta2) * g * g
    mh = m / (1.0 - beta1 ** step)
    vh = v / (1.0 - beta2 ** step)
    x = np.maximum(x - lr * mh / (np.sqrt(vh) + eps), xmin)
    return x, m, v


def update(eps_r, sigma, g_eps, g_sig, state, step, lr_eps, lr_sig, beta1=0.9, beta2=0.999, adam_eps=1e-8,
           tv_iters=10, tv_rho=1.0, tv_lambda=0.01, tv_alpha=1.0, mask_rows=0, eps_min=1.0, sig_min=0.0):
    """One epilogue step; `state` = dict of m_eps, v_eps, m_sig, v_sig (float64 arrays)."""
    out = {}
    for name, x, g, lr, xmin in (("eps", eps_r, g_eps, lr_eps, eps_min), ("sig", sigma, g_sig, lr_sig, sig_min)):
        x = np.asarray(x, dtype=np.float64)
        g = np.asarray(g, dtype=np.float64).copy()
        if tv_iters > 0:
            g += tv_gradient(x, tv_iters, tv_rho, tv_lambda, tv_alpha)
        xn, m, v = adam_step(x, g, state["m_" + name], state["v_" + name], step, lr, beta1, beta2, adam_eps,
                             mask_rows, xmin)
        out[name] = (xn, g)
        state["m_" + name], state["v_" + name] = m, v
    return out["eps"][0], out["sig"][0], out["eps"][1], out["sig"][1]


def lowpass(x, taps):
    """Zero-phase FIR along axis 1 of x[nseries][nt][...] (multiscale stages):
    out[n] = sum_k taps[k] x[n + k - (ntaps-1)/2], zero outside.  Pin: equals np.convolve(..., 'same')
    for symmetric taps; a constant series keeps its value away from the ends when sum(taps) = 1."""
    x = np.asarray(x, dtype=np.float64)
    taps = np.asarray(taps, dtype=np.float64)
    half = (len(taps) - 1) // 2
    out = np.zeros_like(x)
    nt = x.shape[1]
    for k, h in enumerate(taps):
        sh = k - half
        lo, hi = max(0, -sh), min(nt, nt - sh)
        if lo < hi:                                   # (taps may be longer than the series)
            out[:, lo:hi] += h * x[:, lo + sh:hi + sh]
    return out


def lowpass_design(dt, f_cut, ntaps=0):
    """Taps of the multiscale stage filter (PAPER.md:529-531 gives no design; reading R21): Hamming-windowed
    sinc with corner f_cut, scaled to unit gain at DC; ntaps <= 0 picks 4 / (f_cut dt) rounded up to odd.
    h[k] = sinc(2 f_cut dt (k - M)) (0.54 - 0.46 cos(2 pi k / (ntaps - 1))), M = (ntaps - 1)/2, h /= sum(h).
    Pin: equals scipy.signal.firwin(ntaps, f_cut, window="hamming", fs=1/dt) (tests/test_oracle_pins.py)."""
    if ntaps <= 0:
        ntaps = int(4.0 / (f_cut * dt)) | 1
    m = (ntaps - 1) / 2.0
    k = np.arange(ntaps, dtype=np.float64)
    h = np.sinc(2.0 * f_cut * dt * (k - m))
    if ntaps > 1:
        h = h * (0.54 - 0.46 * np.cos(2.0 * np.pi * k / (ntaps - 1)))
    return h / h.sum()


# ------------------------------------------------------------------------------------------------
# Coarser grid for the early multiscale stages ("early-stage use of coarse grids and
# low-frequency data"; the paper gives no transfer operators -- reading R23): node-aligned 2:1 coarsening,
# coarse node (J, I) = fine node (2J, 2I); n_c = (n + 1) // 2 nodes per axis.
# ------------------------------------------------------------------------------------------------
def _w121(n, nc):
    """[nc][n] full-weighting matrix along one axis: (1/4, 1/2, 1/4) around fine node 2J, the weight of a
    neighbour outside the grid folded onto the centre (so rows sum to 1 and constants are kept)."""
    w = np.zeros((nc, n))
    for J in range(nc):
        c = 2 * J
        w[J, c] += 0.5
        for nb in (c - 1, c + 1):
            w[J, nb if 0 <= nb < n else c] += 0.25
    return w


def restrict(fine):
    """Full-weighting restriction of a node-centred model [nz][nx] -> [(nz+1)//2][(nx+1)//2]: the tensor
    product of (1/4, 1/2, 1/4) stencils centred on the fine nodes (2J, 2I)."""
    fine = np.asarray(fine, dtype=np.float64)
    nz, nx = fine.shape
    return _w121(nz, (nz + 1) // 2) @ fine @ _w121(nx, (nx + 1) // 2).T


def _interp(n, nc):
    """[n][nc] linear interpolation along one axis: even fine nodes copy coarse node j/2, odd ones average
    their two coarse neighbours (the last node of an even-sized axis copies the last coarse node)."""
    p = np.zeros((n, nc))
    for j in range(n):
        if j % 2 == 0:
            p[j, j // 2] = 1.0
        else:
            lo, hi = j // 2, min(j // 2 + 1, nc - 1)
            p[j, lo] += 0.5
            p[j, hi] += 0.5
    return p


def prolong(coarse, nz, nx):
    """Bilinear prolongation [nzc][nxc] -> [nz][nx] (the transfer back of a coarse-stage model update)."""
    coarse = np.asarray(coarse, dtype=np.float64)
    return _interp(nz, coarse.shape[0]) @ coarse @ _interp(nx, coarse.shape[1]).T
