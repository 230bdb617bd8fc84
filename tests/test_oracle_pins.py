"""Pins for the float64 oracle: what physics and mathematics fix, independent of any code of ours.

Each test names the pin of DESIGN.md section 6 (after SURVEY.md section 8(c) C.7) it implements and
the mistake it is meant to catch.  None of these re-types the oracle's formula as its own check:
the expectations are an analytic solution (Hankel function via SciPy), conservation laws, symmetry
(reciprocity), the adjoint identity against complex-step derivatives of the forward code, finite
differences of the misfit, closed-form special cases and brute force on tiny inputs.
"""
import os

import numpy as np
import pytest
from scipy.special import hankel2

import gpr_inputs as gi
import oracle
from helpers import problem, rel_l2

C0, MU0, EPS0 = gi.C0, gi.MU0, gi.EPS0


# ------------------------------------------------------------------------------------------------
# Pin 1: analytic 2-D line source  (forward scheme, source scale and sign, time alignment, CPML)
# ------------------------------------------------------------------------------------------------
def _analytic_trace(w, dt, rho, eps_r, sigma, mu_r=1.0):
    """Ez(rho, t_n = n dt) for a z-directed line current I(t) sampled as w[n] = I((n+1/2) dt) in a
    homogeneous medium: Ez(w) = -(w mu0 / 4) I(w) H0^(2)(k rho), k = w sqrt(mu0 eps (1 - j s/(w eps)))
    (Harrington, Time-Harmonic EM Fields, eq. 5-84), e^{+jwt} convention."""
    nt = len(w)
    nfft = 8 * nt
    W = np.fft.rfft(w, nfft)
    om = 2.0 * np.pi * np.fft.rfftfreq(nfft, dt)
    E = np.zeros_like(W)
    o = om[1:]
    eps = EPS0 * eps_r
    mu = MU0 * mu_r
    k = o * np.sqrt(mu * eps * (1.0 - 1j * sigma / (o * eps)))
    k = np.where(k.imag > 0, -k, k)              # decaying branch for e^{+jwt}
    E[1:] = -(o * mu / 4.0) * W[1:] * np.exp(-1j * o * dt / 2.0) * hankel2(0, k * rho)
    return np.fft.irfft(E, nfft)[:nt]


def _line_source_error(dx, eps_r, sigma, offsets_m, mu_r=None):
    f = 400e6
    dt = 2e-11 * dx / 0.01
    nt = int(round(12e-9 / dt))
    npml = int(round(0.2 / dx))
    n = int(round(1.4 / dx)) + 2 * npml + 1
    c = n // 2
    order, smax, kmax, amax = gi.cpml_defaults(dx, f, eps_r)
    w = gi.ricker(nt, dt, f).astype(np.float64)
    recs = []
    for off in offsets_m:
        k = int(round(off / dx))
        recs.append((c, c + k))                    # on-axis
        kd = int(round(off / dx / np.sqrt(2)))
        recs.append((c + kd, c + kd))              # diagonal
    pb = oracle.Problem(nz=n, nx=n, dx=dx, dt=dt, nt=nt, npml=npml, pml_order=order, pml_sigma_max=smax,
                        pml_kappa_max=kmax, pml_alpha_max=amax, src_zx=np.array([[c, c]]),
                        rec_zx=np.array([recs]), wavelet=w)
    tr = oracle.forward(pb, np.full((n, n), eps_r), np.full((n, n), sigma),
                        mu_r=None if mu_r is None else np.full((n, n), mu_r))["traces"][0]
    errs = []
    for r, (z, x) in enumerate(recs):
        rho = dx * np.hypot(z - c, x - c)
        errs.append(rel_l2(tr[:, r], _analytic_trace(w, dt, rho, eps_r, sigma, 1.0 if mu_r is None else mu_r)))
    return np.array(errs)


@pytest.mark.parametrize("eps_r,sigma", [(1.0, 0.0), (4.0, 5e-3)])
def test_pin1_line_source_green_function_second_order(eps_r, sigma):
    """A wrong source scale/sign, a half-step time misalignment, a missing Cb factor or a reflecting
    CPML all give O(1) or O(dt) errors here; the correct scheme converges with order 2."""
    offs = (0.2, 0.4, 0.6)
    e1 = _line_source_error(0.01, eps_r, sigma, offs)
    e2 = _line_source_error(0.005, eps_r, sigma, offs)
    bound = 5e-3 if eps_r == 1.0 else 4e-2      # grid dispersion grows with sqrt(eps_r) at fixed dx
    assert np.all(e1 < bound), e1
    ratio = e1 / e2
    assert np.all(ratio > 3.0) and np.all(ratio < 5.0), (e1, e2, ratio)


# ------------------------------------------------------------------------------------------------
# Pin 2: discrete energy conservation in a lossless PEC box (signs, staggering, ring)
# ------------------------------------------------------------------------------------------------
def test_pin2_energy_conserved_lossless_pec_box():
    wl = gi.small_random(nz=40, nx=46, nt=600, npml=0, nshots=1, nrec=1, lossy=False, seed=7)
    w = wl.wavelet.astype(np.float64).copy()
    nsrc_on = 380
    w[nsrc_on:] = 0.0                              # source switched off after step nsrc_on - 1
    pb = problem(wl, wavelet=w)
    out = oracle.forward(pb, wl.eps_r, wl.sigma, want_h_hist=True)
    ez, hx, hy = out["ez_hist"][0], out["hx_hist"][0], out["hy_hist"][0]
    eps = EPS0 * wl.eps_r.astype(np.float64)
    dx2 = wl.dx ** 2
    ns = np.arange(nsrc_on + 1, wl.nt)             # hx[n] = Hx^{n-1/2}, hx[n+1] = Hx^{n+1/2}
    W = np.array([0.5 * np.sum(eps * ez[n] ** 2) * dx2
                  + 0.5 * MU0 * (np.sum(hx[n + 1] * hx[n]) + np.sum(hy[n + 1] * hy[n])) * dx2 for n in ns])
    assert W[0] > 0
    assert np.max(np.abs(W / W[0] - 1.0)) < 1e-12


# ------------------------------------------------------------------------------------------------
# Pin 3: reciprocity (Cb source factor, collocated materials, H-located CPML tables)
# ------------------------------------------------------------------------------------------------
def test_pin3_reciprocity_heterogeneous_lossy_cpml():
    wl = gi.small_random(nz=60, nx=70, nt=400, npml=10, nshots=1, nrec=1, seed=11)
    a, b = (14, 17), (41, 55)                      # both interior, one close to the CPML
    tr = []
    for s, r in ((a, b), (b, a)):
        pb = problem(wl, src_zx=np.array([s]), rec_zx=np.array([[r]]))
        tr.append(oracle.forward(pb, wl.eps_r, wl.sigma)["traces"][0, :, 0])
    assert np.linalg.norm(tr[0]) > 0
    assert rel_l2(tr[0], tr[1]) < 1e-12



# ------------------------------------------------------------------------------------------------
# Pin 4: adjoint identity <J dm, y> = <dm, J^T y> with J dm from a complex step of the forward code
# ------------------------------------------------------------------------------------------------
def test_pin4_adjoint_identity_complex_step():
    wl = gi.small_random(nz=44, nx=52, nt=160, npml=8, nshots=2, nrec=6, seed=21)
    pb = problem(wl)
    rng = np.random.default_rng(5)
    de = rng.standard_normal((wl.nz, wl.nx))
    ds = rng.standard_normal((wl.nz, wl.nx)) * 1e-2
    y = rng.standard_normal((wl.nshots, wl.nt, wl.nrec))
    h = 1e-30
    trz = oracle.forward(pb, wl.eps_r + 1j * h * de, wl.sigma + 1j * h * ds)["traces"]
    Jdm = trz.imag / h
    ge, gs = oracle.gradient(pb, wl.eps_r, wl.sigma, y)
    lhs = float(np.sum(Jdm * y))
    rhs = float(np.sum(ge * de) + np.sum(gs * ds))
    assert abs(lhs) > 0
    assert abs(lhs - rhs) / abs(lhs) < 1e-10
    # each parameter separately (a swapped chain-rule term would cancel only in the sum by accident)
    Je = oracle.forward(pb, wl.eps_r + 1j * h * de, wl.sigma.astype(np.complex128))["traces"].imag / h
    Js = oracle.forward(pb, wl.eps_r.astype(np.complex128), wl.sigma + 1j * h * ds)["traces"].imag / h
    assert abs(np.sum(Je * y) - np.sum(ge * de)) / abs(np.sum(Je * y)) < 1e-10
    assert abs(np.sum(Js * y) - np.sum(gs * ds)) / abs(np.sum(Js * y)) < 1e-10


# ------------------------------------------------------------------------------------------------
# Pin 5: central finite differences of the misfit (independent of complex arithmetic)
# ------------------------------------------------------------------------------------------------
def test_pin5_finite_differences_of_misfit():
    wl = gi.small_random(nz=44, nx=52, nt=200, npml=8, nshots=1, nrec=6, seed=33)
    pb = problem(wl)
    eps = wl.eps_r.astype(np.float64)
    sig = wl.sigma.astype(np.float64)
    rng = np.random.default_rng(9)
    d_obs = oracle.forward(pb, eps * (1 + 0.05 * rng.standard_normal(eps.shape)), sig * 1.1)["traces"]

    def misfit(e, s):
        return 0.5 * np.sum((oracle.forward(pb, e, s)["traces"] - d_obs) ** 2)

    res = oracle.forward(pb, eps, sig)["traces"] - d_obs
    ge, gs = oracle.gradient(pb, eps, sig, res)
    sz, sx = map(int, wl.src_zx[0])
    cells = [(20, 25), (sz, sx), (3, 30), (22, 2), (30, 40)]     # interior, source, CPML z, CPML x
    for (j, i) in cells:
        for which, g, h in (("eps", ge, 1e-4), ("sig", gs, 1e-6)):
            ep, em, sp, sm = eps.copy(), eps.copy(), sig.copy(), sig.copy()
            if which == "eps":
                ep[j, i] += h; em[j, i] -= h
            else:
                sp[j, i] += h; sm[j, i] -= h
            fd = (misfit(ep, sp) - misfit(em, sm)) / (2 * h)
            assert abs(fd - g[j, i]) <= 2e-6 * max(abs(fd), np.max(np.abs(g)) * 1e-3), (j, i, which, fd, g[j, i])
    # ring cells are never updated: gradient exactly zero there
    for g in (ge, gs):
        assert np.all(g[0, :] == 0) and np.all(g[-1, :] == 0) and np.all(g[:, 0] == 0) and np.all(g[:, -1] == 0)
    # random direction
    de = rng.standard_normal(eps.shape)
    ds = rng.standard_normal(eps.shape) * 1e-3
    h = 1e-5
    fd = (misfit(eps + h * de, sig + h * ds) - misfit(eps - h * de, sig - h * ds)) / (2 * h)
    an = np.sum(ge * de) + np.sum(gs * ds)
    assert abs(fd - an) / abs(an) < 1e-7


# ------------------------------------------------------------------------------------------------
# Pin 6: special cases of the coefficient build and of the CPML tables
# ------------------------------------------------------------------------------------------------
def test_pin6_coefficients_special_cases():
    dt = 2e-11
    er = np.array([1.0, 4.0, 9.5, 20.0])
    # sigma = 0: exactly Eq. (3)'s coefficients: 1 and dt/eps
    ca, cb = oracle.coefficients(er, np.zeros(4), dt)
    assert np.all(ca == 1.0)
    np.testing.assert_allclose(cb, dt / (EPS0 * er), rtol=1e-15)
    # lossy: Ca = (2 eps - sigma dt)/(2 eps + sigma dt), Cb = 2 dt/(2 eps + sigma dt)  (Taflove 3.31)
    sg = np.array([1e-3, 5e-3, 2e-2, 30e-3])
    ca, cb = oracle.coefficients(er, sg, dt)
    e = EPS0 * er
    np.testing.assert_allclose(ca, (2 * e - sg * dt) / (2 * e + sg * dt), rtol=1e-14)
    np.testing.assert_allclose(cb, 2 * dt / (2 * e + sg * dt), rtol=1e-14)
    # first-order agreement with Eq. (3)'s explicit form: Ca = 1 - sigma dt/eps + O((sigma dt/eps)^2)
    x = sg * dt / e
    assert np.all(np.abs(ca - (1 - x)) < x ** 2)
    # sigma > 100 S/m: PEC
    ca, cb = oracle.coefficients(np.array([4.0, 4.0]), np.array([100.0, 100.5]), dt)
    assert ca[1] == 0 and cb[1] == 0 and ca[0] != 0 and cb[0] != 0


def test_pin6_cpml_tables():
    n, P, m, dt = 64, 10, 3, 2e-11
    smax, kmax, amax = 5.0, 3.0, 0.02
    b, c, ik = oracle.cpml_profile(n, P, m, smax, kmax, amax, dt, 0)
    # interior and interface: trivial; symmetric; graded monotonically; ring has rho = 1
    assert np.all(b[P:n - P] == 0) and np.all(c[P:n - P] == 0) and np.all(ik[P:n - P] == 1)
    np.testing.assert_allclose(b, b[::-1], rtol=1e-14)
    np.testing.assert_allclose(c, c[::-1], rtol=1e-14)
    assert np.all(np.diff(ik[:P + 1]) > 0) and abs(ik[0] - 1 / kmax) < 1e-15
    assert abs(b[0] - np.exp(-(smax / kmax) * dt / EPS0)) < 1e-15       # alpha(rho=1) = 0
    assert np.all(c[:P] < 0) and np.all((b[:P] > 0) & (b[:P] < 1))
    bh, ch, ikh = oracle.cpml_profile(n, P, m, smax, kmax, amax, dt, 1)
    assert len(bh) == n - 1
    np.testing.assert_allclose(bh, bh[::-1], rtol=1e-14)
    assert np.all(bh[P:n - 1 - P] == 0) and bh[P - 1] > 0 and bh[n - 1 - P] > 0
    rho = 0.5 / P                                                        # innermost H node
    sp, kap, al = smax * rho ** m, 1 + (kmax - 1) * rho ** m, amax * (1 - rho)
    assert abs(bh[P - 1] - np.exp(-(sp / kap + al) * dt / EPS0)) < 1e-15
    assert abs(ch[P - 1] - sp * (bh[P - 1] - 1) / (kap * (sp + kap * al))) < 1e-18
    # P = 0: all trivial
    b0, c0, ik0 = oracle.cpml_profile(n, 0, m, smax, kmax, amax, dt, 0)
    assert np.all(b0 == 0) and np.all(c0 == 0) and np.all(ik0 == 1)


def test_pin6_npml0_matches_plain_numpy_yee():
    """With no CPML the oracle must equal a psi-free vectorised Yee loop written directly from
    Eqs. (3)-(5) in the Ca/Cb form."""
    wl = gi.small_random(nz=30, nx=36, nt=150, npml=0, nshots=1, nrec=4, seed=3)
    pb = problem(wl)
    tr = oracle.forward(pb, wl.eps_r, wl.sigma)["traces"][0]
    eps = EPS0 * wl.eps_r.astype(np.float64)
    sg = wl.sigma.astype(np.float64)
    dt, dx = wl.dt, wl.dx
    ca = (2 * eps - sg * dt) / (2 * eps + sg * dt)
    cb = 2 * dt / (2 * eps + sg * dt)
    ez = np.zeros((wl.nz, wl.nx)); hx = np.zeros((wl.nz - 1, wl.nx)); hy = np.zeros((wl.nz, wl.nx - 1))
    ref = np.zeros((wl.nt, wl.nrec))
    sz, sx = wl.src_zx[0]
    for n in range(wl.nt):
        ref[n] = ez[wl.rec_zx[0, :, 0], wl.rec_zx[0, :, 1]]
        hx -= dt / MU0 * (ez[1:, :] - ez[:-1, :]) / dx
        hy += dt / MU0 * (ez[:, 1:] - ez[:, :-1]) / dx
        ez[1:-1, 1:-1] = ca[1:-1, 1:-1] * ez[1:-1, 1:-1] + cb[1:-1, 1:-1] * (
            (hy[1:-1, 1:] - hy[1:-1, :-1]) / dx - (hx[1:, 1:-1] - hx[:-1, 1:-1]) / dx)
        ez[sz, sx] -= cb[sz, sx] * float(wl.wavelet[n]) / dx ** 2
    assert np.linalg.norm(ref) > 0
    assert rel_l2(tr, ref) < 1e-13


# ------------------------------------------------------------------------------------------------
# Pin 7: CPML quality against a box so large that no reflection can return
# ------------------------------------------------------------------------------------------------
def test_pin7_cpml_vs_big_box():
    wl = gi.config1(nt=500)
    pb = problem(wl)
    tr = oracle.forward(pb, wl.eps_r, wl.sigma)["traces"]
    # slowest medium eps_r = 4 -> c/2; round trip to the new wall must exceed nt*dt
    pad = int(np.ceil(0.5 * (C0 / 2.0) * wl.nt * wl.dt / wl.dx)) + 5
    eps_b = np.pad(wl.eps_r, pad, mode="edge")
    sig_b = np.pad(wl.sigma, pad, mode="edge")
    pbb = problem(wl, nz=wl.nz + 2 * pad, nx=wl.nx + 2 * pad, npml=0, src_zx=wl.src_zx + pad,
                  rec_zx=wl.rec_zx + pad)
    trb = oracle.forward(pbb, eps_b, sig_b)["traces"]
    err = rel_l2(tr, trb)
    assert err < 5e-4, err            # a sign error in any psi gives growth or >> 1e-2
    # without CPML the same small box reflects strongly: the layer is what makes the difference
    tr0 = oracle.forward(problem(wl, npml=0), wl.eps_r, wl.sigma)["traces"]
    assert rel_l2(tr0, trb) > 50 * err


# ------------------------------------------------------------------------------------------------
# Pin 8: linearity in the wavelet, shot independence, additivity of the gradient over shots
# ------------------------------------------------------------------------------------------------
def test_pin8_linearity_and_shot_independence():
    wl = gi.small_random(nz=40, nx=48, nt=140, npml=8, nshots=3, nrec=5, seed=41)
    rng = np.random.default_rng(2)
    w1 = rng.standard_normal((3, wl.nt))
    w2 = rng.standard_normal((3, wl.nt))
    f = lambda w: oracle.forward(problem(wl, wavelet=w), wl.eps_r, wl.sigma)["traces"]
    assert rel_l2(f(2.0 * w1 - 3.0 * w2), 2.0 * f(w1) - 3.0 * f(w2)) < 1e-13
    full = f(w1)
    res = rng.standard_normal(full.shape)
    ge, gs = oracle.gradient(problem(wl, wavelet=w1), wl.eps_r, wl.sigma, res)
    ge_sum = np.zeros_like(ge); gs_sum = np.zeros_like(gs)
    for s in range(3):
        pbs = problem(wl, wavelet=w1[s], src_zx=wl.src_zx[s:s + 1], rec_zx=wl.rec_zx[s:s + 1])
        assert rel_l2(oracle.forward(pbs, wl.eps_r, wl.sigma)["traces"][0], full[s]) < 1e-15
        a, b = oracle.gradient(pbs, wl.eps_r, wl.sigma, res[s:s + 1])
        ge_sum += a; gs_sum += b
    assert rel_l2(ge_sum, ge) < 1e-13 and rel_l2(gs_sum, gs) < 1e-13


def test_pin8_coincident_receivers_sum():
    wl = gi.small_random(nz=36, nx=40, nt=100, npml=6, nshots=1, nrec=3, seed=43)
    rec = wl.rec_zx.copy()
    rec[0, 2] = rec[0, 0]                           # receivers 0 and 2 on the same node
    rng = np.random.default_rng(3)
    res = rng.standard_normal((1, wl.nt, 3))
    ge, gs = oracle.gradient(problem(wl, rec_zx=rec), wl.eps_r, wl.sigma, res)
    res2 = res[:, :, :2].copy()
    res2[:, :, 0] += res[:, :, 2]
    ge2, gs2 = oracle.gradient(problem(wl, rec_zx=rec[:, :2]), wl.eps_r, wl.sigma, res2)
    assert rel_l2(ge, ge2) < 1e-13 and rel_l2(gs, gs2) < 1e-13


# ------------------------------------------------------------------------------------------------
# Pin 9: checkpoint-and-recompute == stored history
# ------------------------------------------------------------------------------------------------
@pytest.mark.parametrize("K", [1, 7, 50, 149, 150, 400])
def test_pin9_checkpointed_gradient_equals_stored_history(K):
    wl = gi.small_random(nz=40, nx=44, nt=150, npml=8, nshots=2, nrec=4, seed=51)
    pb = problem(wl)
    rng = np.random.default_rng(4)
    res = rng.standard_normal((wl.nshots, wl.nt, wl.nrec))
    ge0, gs0, tr0 = oracle.gradient(pb, wl.eps_r, wl.sigma, res, 0, want_traces=True)
    ge, gs, tr = oracle.gradient(pb, wl.eps_r, wl.sigma, res, K, want_traces=True)
    assert np.array_equal(tr, tr0)
    assert rel_l2(ge, ge0) < 1e-14 and rel_l2(gs, gs0) < 1e-14
    assert rel_l2(tr0, oracle.forward(pb, wl.eps_r, wl.sigma)["traces"]) == 0.0


# ------------------------------------------------------------------------------------------------
# argument checking
# ------------------------------------------------------------------------------------------------
def test_geometry_on_ring_rejected():
    wl = gi.small_random(nz=30, nx=30, nt=10, npml=4, nshots=1, nrec=1)
    with pytest.raises(ValueError):
        oracle.forward(problem(wl, src_zx=np.array([[0, 5]])), wl.eps_r, wl.sigma)
    with pytest.raises(ValueError):
        oracle.forward(problem(wl, rec_zx=np.array([[[5, wl.nx - 1]]])), wl.eps_r, wl.sigma)


# ------------------------------------------------------------------------------------------------
# iteration epilogue (a7): oracle/epilogue.py
# ------------------------------------------------------------------------------------------------
def test_epilogue_adam_first_step_closed_form_mask_and_clamp():
    """Eqs. (14)-(15), at t = 1: m_hat = g, v_hat = g^2, so the step is
    -lr g / (|g| + eps); masked rows do not move; clamps hold."""
    from oracle import epilogue as ep
    rng = np.random.default_rng(3)
    x = rng.uniform(1.0, 9.0, (12, 17)); g = rng.standard_normal((12, 17)) * 3.0
    xn, m, v = ep.adam_step(x, g, np.zeros_like(x), np.zeros_like(x), 1, lr=0.05, eps=1e-8, mask_rows=4, xmin=1.0)
    want = x - 0.05 * g / (np.abs(g) + 1e-8)
    assert np.array_equal(xn[:4], x[:4])
    assert np.allclose(xn[4:], np.maximum(want[4:], 1.0), rtol=0, atol=1e-12)
    assert xn.min() >= 1.0
    # second step against the recursion written out
    g2 = rng.standard_normal(x.shape)
    xn2, m2, v2 = ep.adam_step(xn, g2, m, v, 2, lr=0.05)
    mm = 0.9 * (0.1 * np.where(np.arange(12)[:, None] < 4, 0, g)) + 0.1 * g2
    vv = 0.999 * (0.001 * np.where(np.arange(12)[:, None] < 4, 0, g) ** 2) + 0.001 * g2 ** 2
    assert np.allclose(xn2, xn - 0.05 * (mm / (1 - 0.81)) / (np.sqrt(vv / (1 - 0.999 ** 2)) + 1e-8), atol=1e-12)


def test_epilogue_tv_converges_to_the_rof_minimiser_closed_form():
    """Algorithm 3 is a split-variable solver of min_U 1/2 |U - U0|^2 + lambda TV(U):
    run long enough it must reach that minimiser, which has a closed form for a two-level periodic
    stripe (plateau lengths L1, L2, two jumps per period): the plateaus move towards each other by
    2 lambda / L1 and 2 lambda / L2.  So tv_grad = alpha (X - s U) -> +alpha s 2 lambda / L1 on the high
    plateau and -alpha s 2 lambda / L2 on the low one.  Checked along x and along z (pins the forward /
    backward differences, the sign of the B update and the shrink threshold lambda / rho in each axis)
    and for two values of rho (the limit does not depend on rho)."""
    from oracle import epilogue as ep
    L1, L2, hi, lo, lam, alpha = 10, 14, 8.0, 2.0, 0.01, 0.7
    x = np.empty((4, L1 + L2)); x[:, :L1] = hi; x[:, L1:] = lo
    for rho in (1.0, 0.5):
        for img in (x, x.T.copy()):
            g = ep.tv_gradient(img, iters=1500, rho=rho, lam=lam, alpha=alpha)
            g = g if img is x else g.T
            assert np.allclose(g[:, :L1], alpha * hi * 2 * lam / L1, rtol=1e-9, atol=0)
            assert np.allclose(g[:, L1:], -alpha * hi * 2 * lam / L2, rtol=1e-9, atol=0)
    # lambda beyond the crossing point (0.75 / (2/L1 + 2/L2) = 2.19 for U0 = X / 8): the minimiser is the
    # mean, tv_grad = alpha (X - mean)
    g = ep.tv_gradient(x, iters=1500, rho=1.0, lam=5.0, alpha=1.0)
    assert np.allclose(g, x - x.mean(), atol=1e-8)


def test_epilogue_tv_invariants():
    """Eq. (17) shrink; constant model => zero TV term; the Jacobi sweeps converge to the solution of
    (I + rho D^T D) U = U0 + rho D^T (Z - B) (dense solve on a tiny periodic grid, Z = B = 0 so U -> the
    screened-Poisson smoothing of U0); TV term is small and acts against roughness."""
    from oracle import epilogue as ep
    vx, vz = ep.shrink(np.array([3.0, 0.1, 0.0]), np.array([4.0, 0.1, 0.0]), 1.0)
    assert np.allclose(vx, [3.0 * 0.8, 0.0, 0.0]) and np.allclose(vz, [4.0 * 0.8, 0.0, 0.0])
    assert np.all(ep.tv_gradient(np.full((9, 11), 7.5)) == 0.0)
    rng = np.random.default_rng(5)
    nz, nx, rho = 6, 7, 1.0
    x = rng.uniform(1, 2, (nz, nx))
    # dense periodic operator I + rho D^T D  (D^T D = 4 I - neighbours)
    n = nz * nx
    A = np.zeros((n, n))
    for j in range(nz):
        for i in range(nx):
            k = j * nx + i
            A[k, k] = 1 + 4 * rho
            for (jj, ii) in ((j, (i + 1) % nx), (j, (i - 1) % nx), ((j + 1) % nz, i), ((j - 1) % nz, i)):
                A[k, jj * nx + ii] -= rho
    s = np.abs(x).max()
    u_exact = np.linalg.solve(A, (x / s).ravel()).reshape(nz, nx)
    # lambda so large that Z stays 0 (everything shrunk away) and B only accumulates G; one iteration = one sweep
    g1 = ep.tv_gradient(x, iters=1, rho=rho, lam=1e9, alpha=1.0)
    u1 = (x - g1) / s
    nb = np.roll(x / s, 1, 0) + np.roll(x / s, -1, 0) + np.roll(x / s, 1, 1) + np.roll(x / s, -1, 1)
    assert np.allclose(u1, (x / s + rho * nb) / (1 + 4 * rho), atol=1e-14)            # the sweep itself
    # fixed point of the sweep with Z = B = 0 frozen is the dense solution
    u = x / s
    for _ in range(200):
        nbu = np.roll(u, 1, 0) + np.roll(u, -1, 0) + np.roll(u, 1, 1) + np.roll(u, -1, 1)
        u = (x / s + rho * nbu) / (1 + 4 * rho)
    assert np.allclose(u, u_exact, atol=1e-10)
    # roughness: TV term correlates positively with (x - local mean)
    g = ep.tv_gradient(x)
    loc = x - 0.25 * (np.roll(x, 1, 0) + np.roll(x, -1, 0) + np.roll(x, 1, 1) + np.roll(x, -1, 1))
    assert np.sum(g * loc) > 0


def test_golden_config1_oracle_values_unchanged():
    """tests/golden/config1_oracle.txt (written by tests/golden/make_golden.py from the oracle alone):
    the oracle and the input generator still give the frozen numbers."""
    import importlib.util
    here = os.path.dirname(os.path.abspath(__file__))
    spec = importlib.util.spec_from_file_location("make_golden", os.path.join(here, "golden", "make_golden.py"))
    mg = importlib.util.module_from_spec(spec); spec.loader.exec_module(mg)
    now = mg.values()
    with open(os.path.join(here, "golden", "config1_oracle.txt")) as f:
        for line in f:
            if line.startswith("#"):
                continue
            k, v = line.rsplit(" ", 1)
            assert abs(now[k] - float(v)) <= 1e-9 * max(abs(float(v)), 1e-30), k


def test_lowpass_oracle_equals_numpy_convolve():
    from oracle import epilogue as ep
    rng = np.random.default_rng(1)
    x = rng.standard_normal((2, 200, 3))
    k = np.arange(31) - 15
    taps = np.sinc(0.2 * k) * np.hamming(31); taps /= taps.sum()
    y = ep.lowpass(x, taps)
    for s in range(2):
        for r in range(3):
            assert np.allclose(y[s, :, r], np.convolve(x[s, :, r], taps, mode="same"), atol=1e-13)
    assert np.allclose(ep.lowpass(np.ones((1, 100, 1)), taps)[0, 20:80, 0], 1.0, atol=1e-13)


# ------------------------------------------------------------------------------------------------
# mu_r model input (Table 1 `miu`; uH4 = dt / (mu0 mu_r); reading R22)
# ------------------------------------------------------------------------------------------------
def test_mu_r_line_source_green_function_second_order():
    """Homogeneous mu_r = 2: the analytic line-source field has mu = mu0 mu_r in BOTH the amplitude
    -(w mu / 4) and the wavenumber; a Db that ignored mu_r, or used it in only one of the two H updates,
    gives O(1) errors (wrong speed / anisotropy), the correct scheme converges with order 2."""
    offs = (0.2, 0.4)
    e1 = _line_source_error(0.01, 2.0, 2e-3, offs, mu_r=2.0)
    e2 = _line_source_error(0.005, 2.0, 2e-3, offs, mu_r=2.0)
    assert np.all(e1 < 4e-2), e1
    ratio = e1 / e2
    assert np.all(ratio > 3.0) and np.all(ratio < 5.0), (e1, e2, ratio)


def _random_mu(wl, seed):
    return np.random.default_rng(seed).uniform(1.0, 3.0, (wl.nz, wl.nx))


def test_mu_r_energy_conserved_with_heterogeneous_permeability():
    """Lossless PEC box, heterogeneous eps_r AND mu_r: the discrete energy with mu0 mu_r[j][i] weighting the
    H component stored at array index (j, i) is conserved to round-off once the source is off.  A mu_r taken
    from a neighbouring index, applied to one H component only, or left out of the CPML-free update breaks
    this at O(1)."""
    wl = gi.small_random(nz=40, nx=46, nt=600, npml=0, nshots=1, nrec=1, lossy=False, seed=8)
    mu = _random_mu(wl, 3)
    w = wl.wavelet.astype(np.float64).copy()
    nsrc_on = 380
    w[nsrc_on:] = 0.0
    out = oracle.forward(problem(wl, wavelet=w), wl.eps_r, wl.sigma, want_h_hist=True, mu_r=mu)
    ez, hx, hy = out["ez_hist"][0], out["hx_hist"][0], out["hy_hist"][0]
    eps = EPS0 * wl.eps_r.astype(np.float64)
    dx2 = wl.dx ** 2
    ns = np.arange(nsrc_on + 1, wl.nt)
    W = np.array([0.5 * np.sum(eps * ez[n] ** 2) * dx2
                  + 0.5 * MU0 * (np.sum(mu[:-1, :] * hx[n + 1] * hx[n]) + np.sum(mu[:, :-1] * hy[n + 1] * hy[n])) * dx2
                  for n in ns])
    assert W[0] > 0
    assert np.max(np.abs(W / W[0] - 1.0)) < 1e-12
    # ... and the same sum with mu_r left out of the weights is NOT constant (the test can fail)
    W1 = np.array([0.5 * np.sum(eps * ez[n] ** 2) * dx2
                   + 0.5 * MU0 * (np.sum(hx[n + 1] * hx[n]) + np.sum(hy[n + 1] * hy[n])) * dx2 for n in ns])
    assert np.max(np.abs(W1 / W1[0] - 1.0)) > 1e-3


def test_mu_r_reciprocity_and_adjoint_identity():
    """Heterogeneous lossy model with CPML and heterogeneous mu_r: swapping source and receiver leaves the
    trace unchanged (1e-12), and <J dm, y> = <dm, J^T y> with J dm from the complex-step forward (1e-10):
    the transpose of the H update carries the same per-cell Db on the same component."""
    wl = gi.small_random(nz=60, nx=70, nt=400, npml=10, nshots=1, nrec=1, seed=12)
    mu = _random_mu(wl, 4)
    a, b = (14, 17), (41, 55)
    tr = []
    for s_, r_ in ((a, b), (b, a)):
        pb = problem(wl, src_zx=np.array([s_]), rec_zx=np.array([[r_]]))
        tr.append(oracle.forward(pb, wl.eps_r, wl.sigma, mu_r=mu)["traces"][0, :, 0])
    assert np.linalg.norm(tr[0]) > 0 and rel_l2(tr[0], tr[1]) < 1e-12
    assert rel_l2(tr[0], oracle.forward(problem(wl, src_zx=np.array([a]), rec_zx=np.array([[b]])), wl.eps_r,
                                        wl.sigma)["traces"][0, :, 0]) > 1e-2       # mu_r does change the answer
    wl = gi.small_random(nz=44, nx=52, nt=160, npml=8, nshots=2, nrec=6, seed=22)
    mu = _random_mu(wl, 5)
    pb = problem(wl)
    rng = np.random.default_rng(6)
    de = rng.standard_normal((wl.nz, wl.nx)); ds = rng.standard_normal((wl.nz, wl.nx)) * 1e-2
    y = rng.standard_normal((wl.nshots, wl.nt, wl.nrec))
    h = 1e-30
    Jdm = oracle.forward(pb, wl.eps_r + 1j * h * de, wl.sigma + 1j * h * ds, mu_r=mu)["traces"].imag / h
    ge, gs = oracle.gradient(pb, wl.eps_r, wl.sigma, y, mu_r=mu)
    lhs, rhs = float(np.sum(Jdm * y)), float(np.sum(ge * de) + np.sum(gs * ds))
    assert abs(lhs) > 0 and abs(lhs - rhs) / abs(lhs) < 1e-10
    ge_k, gs_k = oracle.gradient(pb, wl.eps_r, wl.sigma, y, checkpoint_stride=37, mu_r=mu)
    assert rel_l2(ge_k, ge) < 1e-13 and rel_l2(gs_k, gs) < 1e-13


def test_mu_r_of_one_is_the_default():
    wl = gi.small_random(nz=44, nx=52, nt=120, npml=8, nshots=2, nrec=5, seed=23)
    pb = problem(wl)
    y = gi.random_residual(wl, 1.0)
    one = np.ones((wl.nz, wl.nx))
    assert np.array_equal(oracle.forward(pb, wl.eps_r, wl.sigma)["traces"],
                          oracle.forward(pb, wl.eps_r, wl.sigma, mu_r=one)["traces"])
    for a_, b_ in zip(oracle.gradient(pb, wl.eps_r, wl.sigma, y), oracle.gradient(pb, wl.eps_r, wl.sigma, y, mu_r=one)):
        assert np.array_equal(a_, b_)


# ------------------------------------------------------------------------------------------------
# multiscale stage filter design and grid transfer operators (readings R21, R23)
# ------------------------------------------------------------------------------------------------
def test_lowpass_design_equals_scipy_firwin():
    """The stage filter's taps against a library routine: scipy.signal.firwin with a Hamming window."""
    from scipy.signal import firwin
    from oracle import epilogue as ep
    for dt, f_cut, ntaps in ((2e-11, 150e6, 0), (1e-10, 80e6, 0), (2e-11, 400e6, 33), (1e-11, 1e9, 1)):
        h = ep.lowpass_design(dt, f_cut, ntaps)
        assert len(h) % 2 == 1 and (ntaps <= 0 or len(h) == ntaps)
        assert abs(h.sum() - 1.0) < 1e-14 and np.allclose(h, h[::-1], atol=1e-16)
        assert np.allclose(h, firwin(len(h), f_cut, window="hamming", fs=1.0 / dt), rtol=1e-12, atol=1e-15)
    assert len(ep.lowpass_design(2e-11, 150e6)) == (int(4.0 / (150e6 * 2e-11)) | 1)


def test_grid_transfer_operators():
    """restrict / prolong (R23): constants and (away from the edges) linear fields are reproduced exactly;
    prolong(restrict(f)) differs from a smooth f by O(h^2) (error / 4 when the grid is refined by 2);
    shapes follow n_c = (n + 1) // 2 on odd and even axes; restrict of a single fine node is the 1-2-1 stencil."""
    from oracle import epilogue as ep
    for nz, nx in ((41, 57), (40, 56), (33, 34)):
        c = ep.restrict(np.full((nz, nx), 3.25))
        assert c.shape == ((nz + 1) // 2, (nx + 1) // 2) and np.allclose(c, 3.25, rtol=0, atol=1e-14)
        assert np.allclose(ep.prolong(c, nz, nx), 3.25, rtol=0, atol=1e-14)
        z, x = np.meshgrid(np.arange(nz, dtype=float), np.arange(nx, dtype=float), indexing="ij")
        lin = 2.0 + 0.3 * z - 0.7 * x
        r = ep.restrict(lin)
        assert np.allclose(r[1:-1, 1:-1], lin[2:-2:2, 2:-2:2][:r.shape[0] - 2, :r.shape[1] - 2], atol=1e-12)
        back = ep.prolong(lin[::2, ::2], nz, nx)            # injection then bilinear: exact for linear fields
        assert np.allclose(back[:2 * (r.shape[0] - 1) + 1, :2 * (r.shape[1] - 1) + 1],
                           lin[:2 * (r.shape[0] - 1) + 1, :2 * (r.shape[1] - 1) + 1], atol=1e-12)
    d = np.zeros((9, 9)); d[4, 4] = 1.0
    assert np.allclose(ep.restrict(d)[1:4, 1:4], np.outer([0, 0.5, 0], [0, 0.5, 0]) + 0, atol=1e-15)
    d[4, 4] = 0.0; d[3, 4] = 1.0                              # an odd fine node feeds its two coarse neighbours
    assert np.allclose(ep.restrict(d)[:, 2], [0, 0.125, 0.125, 0, 0], atol=1e-15)
    errs = []
    for n in (33, 65, 129):
        t = np.linspace(0.0, 1.0, n)
        f = np.sin(2 * np.pi * t)[:, None] * np.cos(3 * np.pi * t)[None, :] + t[:, None] ** 2
        e = ep.prolong(ep.restrict(f), n, n) - f
        errs.append(np.abs(e[4:-4, 4:-4]).max())
    assert 3.3 < errs[0] / errs[1] < 4.7 and 3.3 < errs[1] / errs[2] < 4.7, errs
