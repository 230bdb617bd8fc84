"""Parity of the CUDA path (through the C-ABI) against the float64 oracle.  Needs a B200.

Tolerances are north_star's: relative L2 <= 1e-4 on traces, <= 1e-3 on each gradient, over the whole
array, with both sides given the same seeded inputs and the SAME residual (oracle traces - oracle
d_obs, or a seeded random residual, rounded to fp32) -- DESIGN.md section 8.
"""
import numpy as np
import pytest
import torch

import gpr_inputs as gi
import oracle
from helpers import problem, rel_l2
from test_boundary import params_of
from paper_2506_20513_b200 import (GprfwiError, Simulation, gprfwi_gradient_host, gprfwi_residual,
                                   gprfwi_workspace_bytes, gprfwi_workspace_bytes_host)

pytestmark = pytest.mark.gpu

# north_star's bars are 1e-4 (traces) and 1e-3 (gradients) over the whole array.  Asserted here: 1e-4 on both
# (measured on B200: traces <= 4e-6, gradients <= 3e-5), and -- because a gradient spans many decades and the
# near-source cells dominate a whole-array norm -- the same relative L2 inside each region a bug could hide in
# (CPML strips, the cells around every tile seam, the ring-adjacent cells, the far field), plus the largest
# absolute error against the largest value.  DESIGN.md section 6 lists the measured per-region numbers.
TOL_TRACE, TOL_GRAD = 1e-4, 1e-4
TOL_REGION, TOL_MAXABS = 1e-3, 1e-4
TILE_OZ, TILE_OX = 28, 120          # owned rows / columns of a tile in the default kernel shape


def dev():
    assert torch.cuda.is_available(), "these tests need a CUDA device"
    return torch.device("cuda:0")


def padded(a, pitch):
    out = np.zeros((a.shape[0], pitch), dtype=np.float32)
    out[:, :a.shape[1]] = a
    return out


def run_gpu(wl, residual=None, pitch=None, budget=0, checkpoint_stride=0):
    pitch = pitch or wl.nx
    p = params_of(wl, pitch=pitch, checkpoint_stride=checkpoint_stride)
    sim = Simulation(p, wl.src_zx, wl.rec_zx, wl.wavelet, dev(), budget_bytes=budget)
    sim.workspace.fill_(0xFF)          # NaN everywhere: the library must not rely on a zeroed workspace
    e = torch.as_tensor(padded(wl.eps_r, pitch), device=dev())
    s = torch.as_tensor(padded(wl.sigma, pitch), device=dev())
    tr = sim.forward(e, s).cpu().numpy().copy()
    ge = gs = None
    if residual is not None:
        r = torch.as_tensor(np.ascontiguousarray(residual, dtype=np.float32), device=dev())
        a, b = sim.adjoint(r)
        torch.cuda.synchronize()
        ge, gs = a.cpu().numpy()[:, :wl.nx].copy(), b.cpu().numpy()[:, :wl.nx].copy()
    plan = dict(sim.plan)
    sim.close()
    return tr, ge, gs, plan


def oracle_all(wl, residual=None, with_obs=False):
    pb = problem(wl)
    tr = oracle.forward(pb, wl.eps_r, wl.sigma)["traces"]
    if residual is None:
        if with_obs:
            residual = tr - oracle.forward(pb, wl.eps_r_obs, wl.sigma_obs)["traces"]
        else:
            residual = gi.random_residual(wl, float(np.sqrt(np.mean(tr ** 2))))
    residual = residual.astype(np.float32)
    ge, gs = oracle.gradient(pb, wl.eps_r, wl.sigma, residual)
    return tr, residual, ge, gs


def regions(wl):
    """Boolean masks of the full grid where a localised error would hide under a whole-array norm."""
    nz, nx, P = wl.nz, wl.nx, wl.npml
    j = np.arange(nz)[:, None] * np.ones((1, nx), dtype=np.int64)
    i = np.ones((nz, 1), dtype=np.int64) * np.arange(nx)[None, :]
    out = {}
    if P > 0:
        out["cpml-top"], out["cpml-bottom"] = j < P, j >= nz - P
        out["cpml-left"], out["cpml-right"] = i < P, i >= nx - P
    dj = np.minimum(j % TILE_OZ, TILE_OZ - j % TILE_OZ)
    di = np.minimum(i % TILE_OX, TILE_OX - i % TILE_OX)
    seam_z = (dj <= 4) & (j >= TILE_OZ - 4) & (j <= (nz - 1) // TILE_OZ * TILE_OZ + 4)
    seam_x = (di <= 4) & (i >= TILE_OX - 4) & (i <= (nx - 1) // TILE_OX * TILE_OX + 4)
    if seam_z.any():
        out["tile-seams-z"] = seam_z
    if seam_x.any():
        out["tile-seams-x"] = seam_x
    out["ring-adjacent"] = (j == 1) | (j == nz - 2) | (i == 1) | (i == nx - 2)
    far = np.ones((nz, nx), bool)                      # farther than a third of the grid from every source and receiver
    rad = max(nz, nx) // 3
    pts = np.concatenate([wl.src_zx.reshape(-1, 2), wl.rec_zx.reshape(-1, 2)])
    for z, x in np.unique(pts, axis=0):
        far[max(z - rad, 0):z + rad + 1, max(x - rad, 0):x + rad + 1] = False
    far &= (j >= P) & (j < nz - P) & (i >= P) & (i < nx - P)
    if far.any():
        out["far-field"] = far
    return out


def region_report(wl, g, g_o, name):
    """rel-L2 of a gradient inside each region and the scaled max-abs error.  Regions where the oracle's
    gradient stays below 1e-5 of its peak are left to the max-abs bound: fp32 sums whose terms are of the
    peak's size cannot resolve such cells relative to themselves (ring-adjacent cells deep in the CPML)."""
    rep = {}
    peak = float(np.abs(g_o).max())
    for key, m in regions(wl).items():
        if np.abs(g_o[m]).max() > 1e-5 * peak:
            rep[key] = rel_l2(g[m], g_o[m])
    rep["max-abs/peak"] = float(np.abs(g.astype(np.float64) - g_o).max() / max(peak, 1e-300))
    print(f"[regions] {wl.name} {name}: " + " ".join(f"{k} {v:.1e}" for k, v in rep.items()))
    return rep


def assert_parity(wl, got, ref, tag="", tol_region=None, tol_maxabs=None):
    tr, ge, gs = got
    tr_o, ge_o, gs_o = ref
    et, ee, es = rel_l2(tr, tr_o), rel_l2(ge, ge_o), rel_l2(gs, gs_o)
    print(f"[parity] {wl.name}{tag}: traces {et:.2e} grad_eps_r {ee:.2e} grad_sigma {es:.2e}")
    assert et <= TOL_TRACE, et
    assert ee <= TOL_GRAD, ee
    assert es <= TOL_GRAD, es
    for name, g, g_o in (("grad_eps_r", ge, ge_o), ("grad_sigma", gs, gs_o)):
        for key, v in region_report(wl, g, g_o, name).items():
            assert v <= ((tol_maxabs or TOL_MAXABS) if key == "max-abs/peak" else (tol_region or TOL_REGION)), (name, key, v)


# ------------------------------------------------------------------------------------------------
def test_config1_traces_and_gradients():
    """BASELINE.json config 1 in full: 120x120, nt=800, d_obs from the model with the disc."""
    wl = gi.config1()
    tr_o, res, ge_o, gs_o = oracle_all(wl, with_obs=True)
    tr, ge, gs, plan = run_gpu(wl, res)
    assert plan["full_history"] == 1
    assert_parity(wl, (tr, ge, gs), (tr_o, ge_o, gs_o))
    assert np.all(tr[:, 0, :] == 0.0)               # sample 0 is recorded before the first update
    for g in (ge, gs):                               # PEC ring: exactly zero gradient
        assert np.all(g[0] == 0) and np.all(g[-1] == 0) and np.all(g[:, 0] == 0) and np.all(g[:, -1] == 0)


def test_config1_end_to_end_residual_on_gpu():
    """GPU forms the residual from its own fp32 traces (little margin: |res|/|trace| ~ 2 %)."""
    wl = gi.config1()
    pb = problem(wl)
    tr_o, res_o, ge_o, gs_o = oracle_all(wl, with_obs=True)
    d_obs = oracle.forward(pb, wl.eps_r_obs, wl.sigma_obs)["traces"].astype(np.float32)
    p = params_of(wl)
    ws = torch.empty(gprfwi_workspace_bytes_host(p), dtype=torch.uint8, device=dev())
    tr = np.zeros((wl.nshots, wl.nt, wl.nrec), dtype=np.float32)
    ge, gs, misfit = gprfwi_gradient_host(p, wl.eps_r, wl.sigma, wl.wavelet, wl.src_zx, wl.rec_zx, d_obs, ws, tr)
    assert rel_l2(tr, tr_o) <= TOL_TRACE
    assert abs(misfit - 0.5 * np.sum(res_o.astype(np.float64) ** 2)) <= 2e-3 * misfit
    ee, es = rel_l2(ge, ge_o), rel_l2(gs, gs_o)
    print(f"[parity] config1 end-to-end: grad_eps_r {ee:.2e} grad_sigma {es:.2e} misfit {misfit:.6e}")
    # north_star's 1e-3: the residual is 1.7 % of the traces here, so the traces' 1e-6 becomes 6e-5 in the residual
    # and about 4e-4 in the gradient; every other test gives both sides the same residual
    assert ee <= 1e-3 and es <= 1e-3


@pytest.mark.parametrize("shape", [(44, 52, 8), (70, 150, 10), (97, 263, 12), (40, 40, 0), (33, 129, 5),
                                   (50, 120, 10), (41, 100, 8), (37, 230, 6)])
def test_small_ragged_grids(shape):
    """Several tiles with ragged tails in x and z, scattered interior sources/receivers
    (incl. receivers inside the CPML), CPML thickness not a multiple of 4, and a PEC box."""
    nz, nx, npml = shape
    wl = gi.small_random(nz=nz, nx=nx, nt=150, npml=npml, nshots=3, nrec=7, seed=nz * 1000 + nx)
    tr_o, res, ge_o, gs_o = oracle_all(wl)
    tr, ge, gs, _ = run_gpu(wl, res, pitch=nx + 5)
    assert_parity(wl, (tr, ge, gs), (tr_o, ge_o, gs_o), f" {shape}")


def test_checkpoint_recompute_matches_stored_history_and_subbatched():
    """SURVEY 8(a) a6 / pin 9: checkpoint-and-recompute (forced stride, then a small budget that also
    forces shot sub-batches) reproduces the stored-history traces bit for bit and its gradients up
    to the regrouping of fp32 partial sums."""
    wl = gi.small_random(nz=64, nx=140, nt=101, npml=10, nshots=5, nrec=6, seed=77)
    tr_o, res, ge_o, gs_o = oracle_all(wl)
    full = run_gpu(wl, res)
    assert full[3]["full_history"] == 1
    assert_parity(wl, full[:3], (tr_o, ge_o, gs_o), " full")
    for K in (1, 7, 100, 101):
        ck = run_gpu(wl, res, checkpoint_stride=K)
        assert ck[3]["full_history"] == 0 and ck[3]["checkpoint_stride"] == K
        # the recomputed Ez planes are bit-identical to the first pass, so the traces are too; the
        # gradient sums are regrouped by the time blocking (register partial sums per launch)
        assert np.array_equal(ck[0], full[0])
        assert rel_l2(ck[1], full[1]) < 1e-5 and rel_l2(ck[2], full[2]) < 1e-5
    p = params_of(wl)
    lo = min(b for b in (gprfwi_workspace_bytes(p, int(full[3]["workspace_bytes"] * f))[0]
                         for f in np.linspace(0.2, 0.9, 15)) if b > 0)
    ck = run_gpu(wl, res, budget=lo)
    print("[plan] small budget:", ck[3])
    assert ck[3]["full_history"] == 0
    assert np.array_equal(ck[0], full[0])
    # sub-batched passes change the shot grouping of the gradient sum, hence rounding order only
    assert rel_l2(ck[1], full[1]) < 1e-5 and rel_l2(ck[2], full[2]) < 1e-5
    assert_parity(wl, ck[:3], (tr_o, ge_o, gs_o), " small-budget")


def test_stored_tail_segments_equal_recompute_bit_for_bit(monkeypatch):
    """a6, hybrid plan: workspace the checkpoint plan leaves unused holds the Ez planes of the last
    segments (written by the forward pass), and the adjoint sweeps those without a recompute sweep.
    Same stride and shot grouping as the pure recompute plan, so traces AND gradients must be
    bit-identical to it; checked with some, all and (sub-batched budgets) whatever segments fit."""
    wl = gi.small_random(nz=64, nx=140, nt=101, npml=10, nshots=5, nrec=6, seed=78)
    tr_o, res, ge_o, gs_o = oracle_all(wl)
    K = 12
    p = params_of(wl, checkpoint_stride=K)
    monkeypatch.setenv("GPRFWI_TAIL", "0")
    nb0, plan0 = gprfwi_workspace_bytes(p, 1 << 40)
    assert plan0["stored_segments"] == 0 and plan0["shots_per_pass"] == wl.nshots
    pure = run_gpu(wl, res, budget=nb0, checkpoint_stride=K)
    assert pure[3]["stored_segments"] == 0
    assert_parity(wl, pure[:3], (tr_o, ge_o, gs_o), " pure recompute")
    monkeypatch.setenv("GPRFWI_TAIL", "1")
    per = (K - 1) * wl.nshots * wl.nz * 160 * 4          # one segment's planes (internal pitch 160)
    nseg = -(-wl.nt // K)
    for want, budget in ((3, nb0 + int(3.5 * per)), (nseg, 1 << 40)):
        hy = run_gpu(wl, res, budget=budget, checkpoint_stride=K)
        print("[plan] stored tail:", hy[3])
        assert hy[3]["full_history"] == 0 and hy[3]["stored_segments"] == want
        assert hy[3]["workspace_bytes"] <= budget
        for a, b in zip(hy[:3], pure[:3]):
            assert np.array_equal(a, b)
    # sub-batched adjoint passes together with stored segments (stride 2: one segment's planes cost
    # less than one more shot in the pass, so budgets exist where both happen)
    p2 = params_of(wl, checkpoint_stride=2)
    monkeypatch.setenv("GPRFWI_TAIL", "0")
    nb2 = gprfwi_workspace_bytes(p2, 1 << 40)[0]
    monkeypatch.setenv("GPRFWI_TAIL", "1")
    seen = 0
    for b in np.linspace(0.3, 0.99, 70) * nb2:
        nb, plan = gprfwi_workspace_bytes(p2, int(b))
        if nb == 0 or plan["shots_per_pass"] == wl.nshots or plan["stored_segments"] == 0:
            continue
        seen += 1
        hy = run_gpu(wl, res, budget=int(b), checkpoint_stride=2)
        monkeypatch.setenv("GPRFWI_TAIL", "0")
        ref = run_gpu(wl, res, budget=int(b), checkpoint_stride=2)
        monkeypatch.setenv("GPRFWI_TAIL", "1")
        print("[plan] sub-batched + stored:", hy[3])
        assert ref[3]["stored_segments"] == 0 and ref[3]["shots_per_pass"] == hy[3]["shots_per_pass"] < wl.nshots
        for a, c in zip(hy[:3], ref[:3]):
            assert np.array_equal(a, c)
        if seen == 2:
            break
    assert seen > 0
    print("[plan] sub-batched plans with stored segments checked:", seen)


def test_batched_equals_per_shot_and_adjoint_reusable():
    wl = gi.small_random(nz=60, nx=136, nt=120, npml=8, nshots=4, nrec=5, seed=5)
    tr_o, res, _, _ = oracle_all(wl)
    p = params_of(wl)
    sim = Simulation(p, wl.src_zx, wl.rec_zx, wl.wavelet, dev())
    e = torch.as_tensor(wl.eps_r, device=dev()); s = torch.as_tensor(wl.sigma, device=dev())
    tr = sim.forward(e, s).cpu().numpy().copy()
    r = torch.as_tensor(res, device=dev())
    g1 = [t.cpu().numpy().copy() for t in sim.adjoint(r)]
    g2 = [t.cpu().numpy().copy() for t in sim.adjoint(2.0 * r)]       # second adjoint, same forward
    assert rel_l2(g2[0], 2.0 * g1[0]) < 1e-6 and rel_l2(g2[1], 2.0 * g1[1]) < 1e-6
    sim.close()
    ge_sum = np.zeros_like(g1[0], dtype=np.float64); gs_sum = np.zeros_like(ge_sum)
    for k in range(wl.nshots):
        one = wl.subset([k])
        t1, a, b, _ = run_gpu(one, res[k:k + 1])
        assert np.array_equal(t1[0], tr[k])                            # shots are independent
        ge_sum += a; gs_sum += b
    assert rel_l2(g1[0], ge_sum) < 1e-5 and rel_l2(g1[1], gs_sum) < 1e-5


def test_coincident_receivers_and_receiver_on_source():
    wl = gi.small_random(nz=50, nx=60, nt=100, npml=8, nshots=2, nrec=4, seed=9)
    wl.rec_zx[0, 3] = wl.rec_zx[0, 0]
    wl.rec_zx[1, 2] = wl.src_zx[1]
    tr_o, res, ge_o, gs_o = oracle_all(wl)
    tr, ge, gs, _ = run_gpu(wl, res)
    assert_parity(wl, (tr, ge, gs), (tr_o, ge_o, gs_o))


def test_pec_cells_and_zero_sigma():
    """sigma > 100 S/m => PEC cell (Ca = Cb = 0, zero gradient); sigma = 0 => Ca = 1 exactly."""
    wl = gi.small_random(nz=48, nx=56, nt=120, npml=8, nshots=1, nrec=5, seed=13, lossy=False)
    wl.sigma[20:24, 30:36] = 1.0e3
    tr_o, res, ge_o, gs_o = oracle_all(wl)
    tr, ge, gs, _ = run_gpu(wl, res)
    assert_parity(wl, (tr, ge, gs), (tr_o, ge_o, gs_o))
    assert np.all(ge[20:24, 30:36] == 0) and np.all(gs[20:24, 30:36] == 0)


def test_residual_kernel_and_errors():
    a = torch.randn(100003, device=dev()); b = torch.randn(100003, device=dev())
    r = torch.empty_like(a); m = torch.zeros(1, dtype=torch.float64, device=dev())
    gprfwi_residual(a, b, r, m)
    torch.cuda.synchronize()
    assert torch.equal(r, a - b)
    assert abs(m.item() - 0.5 * float(((a - b).double() ** 2).sum())) < 1e-9 * m.item()
    wl = gi.small_random(nz=30, nx=30, nt=10, npml=4, nshots=1, nrec=1)
    wl.src_zx[0] = (0, 5)
    with pytest.raises(GprfwiError) as ei:
        run_gpu(wl)
    assert ei.value.code == -3                                          # EGEOM
    with pytest.raises(TypeError):
        sim = Simulation(params_of(gi.small_random()), np.zeros((2, 2)), np.zeros((2, 5, 2)), np.zeros(120), dev())
        sim.forward(torch.zeros(44, 52), torch.zeros(44, 52))          # CPU tensors are refused


def test_config2_subset_against_oracle():
    """Config 2 at full grid size and nt, first / middle / last shot (the oracle's full run of 20
    shots is what bench.py times; here 3 shots keep the test in tens of seconds)."""
    wl = gi.config2().subset([0, 10, 19])
    tr_o, res, ge_o, gs_o = oracle_all(wl, with_obs=True)
    tr, ge, gs, _ = run_gpu(wl, res)
    assert_parity(wl, (tr, ge, gs), (tr_o, ge_o, gs_o))


def test_config2_full_launch_configuration_properties():
    """Config 2 exactly as bench.py launches it (20 shots, nt=3000, full history in HBM): the three
    oracle-checked shots must be reproduced bit-for-bit inside the batch (shots are independent),
    and the batched gradient must equal the sum of per-shot gradients."""
    wl = gi.config2()
    sub = wl.subset([0, 10, 19])
    tr_o, res_sub, _, _ = oracle_all(sub, with_obs=True)
    res = gi.random_residual(wl, float(np.sqrt(np.mean(tr_o ** 2))))
    res[[0, 10, 19]] = res_sub
    tr, ge, gs, plan = run_gpu(wl, res)
    assert plan["full_history"] == 1 and plan["shots_per_pass"] == 20
    assert rel_l2(tr[[0, 10, 19]], tr_o) <= TOL_TRACE
    t3, _, _, _ = run_gpu(sub)
    assert np.array_equal(t3, tr[[0, 10, 19]])
    ge_sum, gs_sum = np.zeros_like(ge, dtype=np.float64), np.zeros_like(gs, dtype=np.float64)
    for k in range(wl.nshots):
        _, a, b, _ = run_gpu(wl.subset([k]), res[k:k + 1])
        ge_sum += a; gs_sum += b
    ea, eb = rel_l2(ge, ge_sum), rel_l2(gs, gs_sum)
    print(f"[additivity] config 2: 20-shot batch vs sum of 20 one-shot runs: grad_eps_r {ea:.1e} grad_sigma {eb:.1e}")
    assert ea < 1e-5 and eb < 1e-5


def test_config3_checkpointed_subset_against_oracle():
    """Config 3 grid (540x1040), nt cut to 600 and 2 shots for the oracle's sake, forced through
    checkpoint-and-recompute as the full config requires."""
    wl = gi.config3(nt=600).subset([0, 59])
    tr_o, res, ge_o, gs_o = oracle_all(wl, with_obs=True)
    tr, ge, gs, plan = run_gpu(wl, res, checkpoint_stride=40)
    assert plan["full_history"] == 0
    assert_parity(wl, (tr, ge, gs), (tr_o, ge_o, gs_o))


def test_config4_grid_subset_against_oracle():
    """Config 4 grid (1060x2060, 30-cell CPML, dx 5 mm, 1.2 GHz), nt cut to 300 and the first / last
    shot for the oracle's sake, through checkpoint-and-recompute with a stride that is not a multiple
    of the time block (ragged launches at segment ends)."""
    wl = gi.config4(nt=300).subset([0, 99])
    tr_o, res, ge_o, gs_o = oracle_all(wl)
    tr, ge, gs, plan = run_gpu(wl, res, checkpoint_stride=37)
    assert plan["full_history"] == 0 and plan["checkpoint_stride"] == 37
    assert_parity(wl, (tr, ge, gs), (tr_o, ge_o, gs_o))


def test_config5_4096_grid_short_run_against_oracle():
    """Config 5's 4096 x 4096 grid (5145 tiles: the one-group / one-lane launch regime; plane offsets of
    the second shot beyond 2^24 cells) for 16 steps, one source in the top-left CPML corner tile and one
    near the bottom-right corner, six receivers within four cells of each source so that 16 steps reach
    them.  Everything the wave has not reached must stay exactly zero."""
    import dataclasses
    wl = gi.config5(n=4096, batch=2, nt=16)
    off = np.array([(2, 0), (0, 3), (-3, -1), (4, 4), (-2, 2), (1, -4)])
    src = np.array([(25, 30), (4060, 4070)])
    wl = gi.with_geometry(wl, src, src[:, None, :] + off[None, :, :], name="config5-4096-short")
    wl = dataclasses.replace(wl, wavelet=np.sin(0.6 * np.arange(16)).astype(np.float32))
    tr_o, res, ge_o, gs_o = oracle_all(wl)
    tr, ge, gs, plan = run_gpu(wl, res)
    assert_parity(wl, (tr, ge, gs), (tr_o, ge_o, gs_o))
    far = np.ones((wl.nz, wl.nx), bool)
    for (j, i) in src:
        far[max(j - 40, 0):j + 41, max(i - 40, 0):i + 41] = False
    assert np.all(ge[far] == 0.0) and np.all(gs[far] == 0.0) and np.all(ge_o[far] == 0.0)


def test_config5_per_shot_receivers_batched():
    """Config 5 (512^2, uniform random eps_r / sigma per cell, every shot its own 64 receivers): a
    batch of 8 in one call, shots 0 and 7 against the oracle, and batched == per-shot bit for bit."""
    wl = gi.config5(n=512, batch=8, nt=250)
    sub = wl.subset([0, 7])
    tr_o, res_sub, ge_o, gs_o = oracle_all(sub)
    t2, ge, gs, _ = run_gpu(sub, res_sub)
    assert_parity(sub, (t2, ge, gs), (tr_o, ge_o, gs_o))
    tr, _, _, plan = run_gpu(wl)
    assert np.array_equal(tr[[0, 7]], t2)
    assert plan["shots_per_pass"] == 8


def test_epilogue_update_matches_numpy_oracle():
    """a7: TV term (Algorithm 3) + mask + Adam + clamps, three consecutive steps, vs oracle/epilogue.py
    (float64).  Tolerances: the TV term is a small difference X - sU of O(s) numbers, so it is compared
    against max|X| (1e-5); the updated models to 1e-5 relative."""
    from oracle import epilogue as ep
    from paper_2506_20513_b200 import gprfwi_update, gprfwi_update_workspace_bytes, make_update_params
    wl = gi.small_random(nz=70, nx=150, nt=10, npml=10, nshots=1, nrec=2, seed=21)
    nz, nx, pitch = wl.nz, wl.nx, wl.nx + 3
    rng = np.random.default_rng(7)
    d = dev()
    eps = wl.eps_r.astype(np.float64); sig = wl.sigma.astype(np.float64)
    st = {k: np.zeros((nz, nx)) for k in ("m_eps", "v_eps", "m_sig", "v_sig")}
    t = lambda a: torch.as_tensor(padded(a.astype(np.float32), pitch), device=d)
    d_eps, d_sig = t(eps), t(sig)
    d_m = [torch.zeros((nz, pitch), device=d) for _ in range(4)]
    ws = torch.empty(gprfwi_update_workspace_bytes(nz, pitch), dtype=torch.uint8, device=d)
    for step in (1, 2, 3):
        ge = rng.standard_normal((nz, nx)) * 1e-3; gs = rng.standard_normal((nz, nx)) * 2.0
        d_ge, d_gs = t(ge), t(gs)
        u = make_update_params(step=step, lr_eps_r=0.05, lr_sigma=2e-4, tv_iters=10, tv_lambda=0.01,
                               mask_rows=wl.npml + 6, eps_r_min=1.0, sigma_min=0.0)
        gprfwi_update(nz, nx, pitch, u, d_eps, d_sig, d_ge, d_gs, d_m[0], d_m[1], d_m[2], d_m[3], ws)
        torch.cuda.synchronize()
        eps, sig, ge_tv, gs_tv = ep.update(eps, sig, ge, gs, st, step, 0.05, 2e-4, tv_iters=10, tv_lambda=0.01,
                                           mask_rows=wl.npml + 6)
        for name, got, want, x in (("eps", d_ge, ge_tv, eps), ("sig", d_gs, gs_tv, sig)):
            err = np.abs(got.cpu().numpy()[:, :nx] - want).max()
            assert err <= 1e-5 * np.abs(x).max() + 1e-6 * np.abs(want).max(), (name, step, err)
        assert rel_l2(d_eps.cpu().numpy()[:, :nx], eps) <= 1e-5
        assert rel_l2(d_sig.cpu().numpy()[:, :nx], sig) <= 1e-5
        assert d_eps.cpu().numpy()[:, :nx].min() >= 1.0 and d_sig.cpu().numpy()[:, :nx].min() >= 0.0
        assert torch.all(d_eps[:, nx:] == 0)                       # pitch padding untouched


def test_epilogue_tv_long_run_reaches_rof_closed_form():
    """The CUDA TV term against mathematics rather than the oracle: run to convergence on a two-level
    periodic stripe it must give +alpha s 2 lambda / L1 and -alpha s 2 lambda / L2 (the ROF minimiser's
    closed form, see tests/test_oracle_pins.py), along x (eps_r plane) and along z (sigma plane)."""
    from paper_2506_20513_b200 import gprfwi_update, gprfwi_update_workspace_bytes, make_update_params
    L1, L2, lam, alpha = 10, 14, 0.01, 0.7
    n = L1 + L2
    ex = np.empty((n, n), np.float32); ex[:, :L1] = 8.0; ex[:, L1:] = 2.0           # stripe along x
    sz = np.empty((n, n), np.float32); sz[:L1, :] = 0.04; sz[L1:, :] = 0.01         # stripe along z
    d = dev()
    d_e, d_s = torch.as_tensor(ex.copy(), device=d), torch.as_tensor(sz.copy(), device=d)
    g_e, g_s = torch.zeros((n, n), device=d), torch.zeros((n, n), device=d)
    st = [torch.zeros((n, n), device=d) for _ in range(4)]
    ws = torch.empty(gprfwi_update_workspace_bytes(n, n), dtype=torch.uint8, device=d)
    u = make_update_params(step=1, lr_eps_r=0.0, lr_sigma=0.0, tv_iters=1500, tv_rho=1.0, tv_lambda=lam,
                           tv_alpha=alpha, mask_rows=0)
    gprfwi_update(n, n, n, u, d_e, d_s, g_e, g_s, st[0], st[1], st[2], st[3], ws)
    torch.cuda.synchronize()
    ge, gs = g_e.cpu().numpy(), g_s.cpu().numpy()
    assert np.array_equal(d_e.cpu().numpy(), ex) and np.array_equal(d_s.cpu().numpy(), sz)      # lr = 0
    assert np.allclose(ge[:, :L1], alpha * 8.0 * 2 * lam / L1, rtol=2e-3)
    assert np.allclose(ge[:, L1:], -alpha * 8.0 * 2 * lam / L2, rtol=2e-3)
    assert np.allclose(gs[:L1, :], alpha * 0.04 * 2 * lam / L1, rtol=2e-3)
    assert np.allclose(gs[L1:, :], -alpha * 0.04 * 2 * lam / L2, rtol=2e-3)


def test_many_receivers_per_tile_and_per_shot_wavelets():
    """More receivers in one tile than the CTA has threads (the per-thread receiver entries overflow
    into the strided loops), receivers on every region row (both words of the row mask), and one
    wavelet per shot (wavelet_per_shot = 1)."""
    wl = gi.small_random(nz=60, nx=100, nt=90, npml=8, nshots=2, nrec=900, seed=41)
    rng = np.random.default_rng(2)
    wav = np.stack([wl.wavelet, 0.5 * np.roll(wl.wavelet, 7)]).astype(np.float32)
    wav[1, :7] = 0.0
    pb = problem(wl, wavelet=wav.astype(np.float64))
    tr_o = oracle.forward(pb, wl.eps_r, wl.sigma)["traces"]
    res = (rng.standard_normal(tr_o.shape) * np.sqrt(np.mean(tr_o ** 2))).astype(np.float32)
    ge_o, gs_o = oracle.gradient(pb, wl.eps_r, wl.sigma, res)
    p = params_of(wl, wavelet_per_shot=1)
    sim = Simulation(p, wl.src_zx, wl.rec_zx, wav, dev())
    tr = sim.forward(torch.as_tensor(wl.eps_r, device=dev()), torch.as_tensor(wl.sigma, device=dev())).cpu().numpy().copy()
    ge, gs = [t.cpu().numpy().copy() for t in sim.adjoint(torch.as_tensor(res, device=dev()))]
    sim.close()
    assert_parity(wl, (tr, ge, gs), (tr_o, ge_o, gs_o), " 900 receivers, per-shot wavelets")


def test_no_receivers_forward_only():
    """nrec = 0: nothing to record or inject; forward and adjoint must still run (zero gradient)."""
    wl = gi.small_random(nz=40, nx=50, nt=30, npml=6, nshots=2, nrec=1, seed=8)
    p = params_of(wl, nrec=0)
    sim = Simulation(p, wl.src_zx, np.zeros((2, 0, 2), np.int32), wl.wavelet, dev())
    sim.forward(torch.as_tensor(wl.eps_r, device=dev()), torch.as_tensor(wl.sigma, device=dev()))
    ge, gs = sim.adjoint(torch.zeros((2, 30, 0), device=dev()))
    torch.cuda.synchronize()
    assert float(ge.abs().max()) == 0.0 and float(gs.abs().max()) == 0.0
    sim.close()


def test_handle_reuse_with_new_geometry():
    """One Simulation (one handle, one workspace) swept over different shot sets, as bench.py does for
    batches that do not fit one call: results must equal those of fresh handles, bit for bit."""
    wl = gi.small_random(nz=64, nx=130, nt=80, npml=8, nshots=4, nrec=6, seed=17)
    a, b = wl.subset([0, 1]), wl.subset([2, 3])
    ra, rb = gi.random_residual(a, 1.0, seed=1), gi.random_residual(b, 1.0, seed=2)
    fresh = [run_gpu(a, ra), run_gpu(b, rb)]
    p = params_of(a)
    sim = Simulation(p, a.src_zx, a.rec_zx, a.wavelet, dev())
    e = torch.as_tensor(wl.eps_r, device=dev()); s = torch.as_tensor(wl.sigma, device=dev())
    for sub, res, ref in ((a, ra, fresh[0]), (b, rb, fresh[1]), (a, ra, fresh[0])):
        sim.src_zx, sim.rec_zx = sub.src_zx, sub.rec_zx
        tr = sim.forward(e, s).cpu().numpy().copy()
        ge, gs = [t.cpu().numpy().copy() for t in sim.adjoint(torch.as_tensor(res, device=dev()))]
        assert np.array_equal(tr, ref[0]) and np.array_equal(ge, ref[1]) and np.array_equal(gs, ref[2])
    sim.close()


def test_two_live_handles_with_and_without_cpml_interleaved():
    """Two handles alive at once, one with a CPML and one PEC box (whose kernels ask for less dynamic shared
    memory), called alternately: the kernels' shared-memory limit is a per-kernel attribute, so neither handle
    may lower it under the other; results must equal those of fresh handles bit for bit."""
    a = gi.small_random(nz=64, nx=130, nt=60, npml=8, nshots=2, nrec=5, seed=91)
    b = gi.small_random(nz=40, nx=40, nt=60, npml=0, nshots=2, nrec=5, seed=92)
    ra, rb = gi.random_residual(a, 1.0, seed=3), gi.random_residual(b, 1.0, seed=4)
    ref = {"a": run_gpu(a, ra), "b": run_gpu(b, rb)}
    sims = {k: Simulation(params_of(w), w.src_zx, w.rec_zx, w.wavelet, dev()) for k, w in (("a", a), ("b", b))}
    models = {k: (torch.as_tensor(w.eps_r, device=dev()), torch.as_tensor(w.sigma, device=dev())) for k, w in (("a", a), ("b", b))}
    for k, res in (("a", ra), ("b", rb), ("a", ra), ("b", rb), ("a", ra)):
        tr = sims[k].forward(*models[k]).cpu().numpy().copy()
        ge, gs = [t.cpu().numpy().copy() for t in sims[k].adjoint(torch.as_tensor(res, device=dev()))]
        assert np.array_equal(tr, ref[k][0]) and np.array_equal(ge, ref[k][1]) and np.array_equal(gs, ref[k][2]), k
    for sm in sims.values():
        sm.close()


def test_inversion_loop_reduces_misfit_and_recovers_anomaly():
    """the whole iteration (forward, residual, adjoint, TV + Adam update) as C-ABI calls.
    Config 1: start from the layered background, observed data from the model with the disc; the
    misfit must fall, masked rows must not move and the clamps must hold.
    (One source and ten surface receivers do not determine the disc: no claim on the recovered image.)"""
    from paper_2506_20513_b200 import invert
    wl = gi.config1()
    pb = problem(wl)
    d_obs = torch.as_tensor(oracle.forward(pb, wl.eps_r_obs, wl.sigma_obs)["traces"].astype(np.float32), device=dev())
    sim = Simulation(params_of(wl), wl.src_zx, wl.rec_zx, wl.wavelet, dev())
    eps = torch.as_tensor(wl.eps_r.copy(), device=dev()); sig = torch.as_tensor(wl.sigma.copy(), device=dev())
    hist = invert(sim, eps, sig, d_obs, iterations=25, lr_eps_r=0.08, lr_sigma=0.0, mask_rows=wl.npml + 8,
                  tv_iters=5, tv_lambda=0.002, tv_alpha=0.0)
    sim.close()
    print("[invert] misfit", " ".join(f"{h:.3e}" for h in hist[::4]))
    assert hist[-1] < 0.6 * hist[0]
    assert min(hist) == min(hist[len(hist) // 2:])            # still improving in the second half (Adam is not monotone)
    d = eps.cpu().numpy() - wl.eps_r
    assert np.all(d[:wl.npml + 8] == 0.0) and np.abs(d[wl.npml + 8:]).max() > 0.0
    assert eps.min().item() >= 1.0 and torch.equal(sig.cpu(), torch.as_tensor(wl.sigma))      # lr_sigma = 0


def test_lowpass_matches_oracle():
    """Multiscale stage filter: zero-phase FIR along time of traces and of a wavelet."""
    from oracle import epilogue as ep
    from paper_2506_20513_b200 import gprfwi_lowpass, gprfwi_lowpass_design
    rng = np.random.default_rng(4)
    x = rng.standard_normal((3, 517, 11)).astype(np.float32)
    taps = gprfwi_lowpass_design(2e-11, 150e6)
    assert np.allclose(taps, ep.lowpass_design(2e-11, 150e6), rtol=2e-7, atol=1e-9)      # library design vs the oracle's
    assert len(taps) % 2 == 1
    d_x = torch.as_tensor(x, device=dev()); d_t = torch.as_tensor(taps, device=dev())
    y = gprfwi_lowpass(d_x, torch.empty_like(d_x), d_t).cpu().numpy()
    assert rel_l2(y, ep.lowpass(x, taps)) <= 1e-6
    w = gi.ricker(800, 2e-11, 400e6)[None, :]
    d_w = torch.as_tensor(w, device=dev())
    yw = gprfwi_lowpass(d_w, torch.empty_like(d_w), d_t).cpu().numpy()
    assert rel_l2(yw, ep.lowpass(w[:, :, None], taps)[:, :, 0]) <= 1e-6
    assert np.abs(np.fft.rfft(yw[0]))[60:].max() < 0.2 * np.abs(np.fft.rfft(w[0])).max()      # highs are gone


def test_crosshole_and_moving_array_acquisitions():
    """the acquisition variants of Table 1 are per-shot receiver lists.
    Cross-hole shapes of section 4.1 (120 x 220 grid, one source, 200 receivers down the
    other hole, so every tile row holds receivers), a moving source-receiver array, and a
    common-offset profile (one receiver per shot)."""
    wl = gi.crosshole(nt=700)
    tr_o, res, ge_o, gs_o = oracle_all(wl, with_obs=True)
    tr, ge, gs, _ = run_gpu(wl, res)
    assert_parity(wl, (tr, ge, gs), (tr_o, ge_o, gs_o))
    base = gi.small_random(nz=64, nx=170, nt=150, npml=8, nshots=1, nrec=1, seed=77)
    for tag, (src, rec) in (("moving array", gi.acquisition((12, 14), (1, 23), 6, (12, 20), (0, 7), 5)),
                            ("common offset", gi.acquisition((11, 12), (0, 15), 10, (11, 18), (0, 0), 1)),
                            ("fixed receivers", gi.acquisition((50, 15), (-3, 28), 5, (10, 10), (2, 9), 16,
                                                               fixed_receiver=True))):
        wl2 = gi.with_geometry(base, src, rec, name="small-random " + tag)
        tr_o, res, ge_o, gs_o = oracle_all(wl2)
        tr, ge, gs, _ = run_gpu(wl2, res)
        assert_parity(wl2, (tr, ge, gs), (tr_o, ge_o, gs_o))


def test_staged_inversion_driver():
    """SURVEY 8(f)-1/-2, reading R21: two-stage learning-rate strategy (eps_r only, then both) with a
    low-passed first stage, on the cross-hole shapes.  Checked against the oracle where the result is
    fixed: the first misfit of each stage equals the oracle's misfit at that stage's starting models
    with that stage's (filtered) wavelet and data; sigma does not move while its rate is 0; the
    filtered stage leaves the full-band wavelet in place afterwards; each stage lowers its misfit."""
    from oracle import epilogue as ep
    from paper_2506_20513_b200 import Stage, invert_staged
    wl = gi.crosshole(nt=600)
    pb = problem(wl)
    d_obs64 = oracle.forward(pb, wl.eps_r_obs, wl.sigma_obs)["traces"]
    d_obs = torch.as_tensor(d_obs64.astype(np.float32), device=dev())
    sim = Simulation(params_of(wl), wl.src_zx, wl.rec_zx, wl.wavelet, dev())
    eps = torch.as_tensor(wl.eps_r.copy(), device=dev()); sig = torch.as_tensor(wl.sigma.copy(), device=dev())
    stages = [Stage(4, 0.05, 0.0, f_cut=80e6), Stage(4, 0.05, 2e-4)]
    snap = {}

    def cb(k, it, mf):
        if it == stages[k].iterations:
            snap[k] = (eps.cpu().numpy().copy(), sig.cpu().numpy().copy())

    hist = invert_staged(sim, eps, sig, d_obs, stages, callback=cb, mask_rows=0, tv_iters=3, tv_lambda=0.002,
                         tv_alpha=0.0)
    assert torch.equal(sim.wavelet.cpu(), torch.as_tensor(wl.wavelet))
    sim.close()
    print("[staged]", [" ".join(f"{h:.3e}" for h in hs) for hs in hist])
    assert [len(h) for h in hist] == [4, 4]
    assert np.array_equal(snap[0][1], wl.sigma) and not np.array_equal(snap[0][0], wl.eps_r)
    assert not np.array_equal(snap[1][1], wl.sigma)
    assert hist[0][-1] < hist[0][0] and hist[1][-1] < hist[1][0]
    taps = ep.lowpass_design(wl.dt, 80e6)          # the oracle's own statement of the stage filter
    w_lp = ep.lowpass(wl.wavelet[None, :, None], taps)[0, :, 0]
    d_lp = ep.lowpass(d_obs.cpu().numpy(), taps)
    r0 = oracle.forward(problem(wl, wavelet=w_lp), wl.eps_r, wl.sigma)["traces"] - d_lp
    assert abs(hist[0][0] - 0.5 * np.sum(r0 * r0)) <= 1e-3 * hist[0][0]
    r1 = oracle.forward(pb, snap[0][0], snap[0][1])["traces"] - d_obs.cpu().numpy()
    assert abs(hist[1][0] - 0.5 * np.sum(r1 * r1)) <= 1e-3 * hist[1][0]


def test_random_shapes_fuzz():
    """Seeded random grids (ragged tiles, nx a multiple of the tile width or one past it, CPML
    thickness 0 / 3 / 4 / 7 / 10 / 13), shot counts, receiver counts and checkpoint strides against the
    oracle.  160 such cases were run during development; 14 are kept here."""
    rng = np.random.default_rng(2025)
    for case in range(14):
        npml = int(rng.choice([0, 3, 4, 7, 10, 13]))
        nz = int(rng.integers(2 * npml + 7, 2 * npml + 100)); nx = int(rng.integers(2 * npml + 7, 2 * npml + 280))
        if case % 5 == 0:
            nx = 120 * int(rng.integers(1, 3)) + int(rng.choice([0, 1, 4]))
        nt = int(rng.integers(60, 140)); S = int(rng.integers(1, 5)); R = int(rng.integers(1, 9))
        K = int(rng.choice([0, 0, 1, 3, 5, 16]))
        wl = gi.small_random(nz=nz, nx=nx, nt=nt, npml=npml, nshots=S, nrec=R, seed=3000 + case)
        tr_o, res, ge_o, gs_o = oracle_all(wl)
        if np.linalg.norm(ge_o) < 1e-20:        # the wave has not reached a receiver yet: nothing to compare
            continue
        tr, ge, gs, _ = run_gpu(wl, res, checkpoint_stride=min(K, nt))
        assert_parity(wl, (tr, ge, gs), (tr_o, ge_o, gs_o), f" fuzz {case}: {nz}x{nx} npml {npml} nt {nt} S {S} R {R} K {K}")


def test_config3_full_launch_configuration_properties():
    """Config 3 exactly as bench.py launches it (60 shots, nt = 4000, checkpoint-and-recompute chosen by
    the plan): shot 0's traces against the oracle, shots 0 and 59 bit-identical to a two-shot run, and
    the full-batch gradient equal to the sum of the gradients of the two half batches."""
    wl = gi.config3()
    free, _ = torch.cuda.mem_get_info(dev())
    budget = int(free * 0.9)
    res = gi.random_residual(wl, 1.0, seed=5)
    tr, ge, gs, plan = run_gpu(wl, res, budget=budget)
    assert plan["full_history"] == 0
    one = wl.subset([0])
    tr_o = oracle.forward(problem(one), one.eps_r, one.sigma)["traces"]
    assert rel_l2(tr[:1], tr_o) <= TOL_TRACE
    sub = wl.subset([0, 59])
    t2, _, _, _ = run_gpu(sub, budget=budget)
    assert np.array_equal(t2, tr[[0, 59]])
    ga, gb = np.zeros_like(ge, dtype=np.float64), np.zeros_like(gs, dtype=np.float64)
    for lo, hi in ((0, 30), (30, 60)):
        half = wl.subset(list(range(lo, hi)))
        _, a, b, _ = run_gpu(half, res[lo:hi], budget=budget)
        ga += a; gb += b
    assert rel_l2(ge, ga) <= 1e-5 and rel_l2(gs, gb) <= 1e-5


# ------------------------------------------------------------------------------------------------
# parity at the sizes bench.py times, in the plans it gets (SURVEY 8(c) "parity protocol":
# a declared subset of shots with ALL nt and the full grid).  The whole batch runs at full nt with a residual
# that is zero except on one shot, so the batch gradient IS that shot's gradient and is compared -- together
# with that shot's traces -- with a one-shot oracle run at full nt.
# ------------------------------------------------------------------------------------------------
def _one_hot_residual_case(wl, shot, budget, oracle_stride, tol_local=None):
    one = wl.subset([shot])
    pb = problem(one)
    rng = np.random.default_rng(1000 + shot)
    res1 = rng.standard_normal((1, wl.nt, wl.nrec)).astype(np.float32)
    res1[:, 0, :] = 0.0
    ge_o, gs_o, tr_o = oracle.gradient(pb, one.eps_r, one.sigma, res1, checkpoint_stride=oracle_stride, want_traces=True)
    res = np.zeros((wl.nshots, wl.nt, wl.nrec), dtype=np.float32)
    res[shot] = res1[0]
    tr, ge, gs, plan = run_gpu(wl, res, budget=budget)
    print(f"[plan] {wl.name} one-hot shot {shot}:", plan)
    assert_parity(one, (tr[shot:shot + 1], ge, gs), (tr_o, ge_o, gs_o), f" full nt, batch of {wl.nshots}, residual on shot {shot}",
                  tol_region=tol_local, tol_maxabs=tol_local)
    return plan


def _bench_budget():
    import gc
    gc.collect()
    torch.cuda.empty_cache()                  # (earlier tests' cached blocks would shrink the plan bench.py gets)
    free, _ = torch.cuda.mem_get_info(dev())
    return int(free * 0.9)


@pytest.mark.parametrize("shot", [0, 59])
def test_config3_full_nt_in_benchmarked_plan_against_oracle(shot):
    """Config 3 as bench.py runs it (60 shots, nt = 4000, the plan the library picks for the free HBM:
    checkpoint-and-recompute with stored tail segments, 3 lanes), first and last shot of the pass."""
    plan = _one_hot_residual_case(gi.config3(), shot, _bench_budget(), oracle_stride=0)
    assert plan["full_history"] == 0 and plan["shots_per_pass"] == 60


def test_config4_full_nt_in_benchmarked_plan_against_oracle():
    """Config 4 as bench.py runs it (100 shots, nt = 6000; sub-batched adjoint passes, K chosen by the plan):
    the LAST shot of the first adjoint pass (the end of a lane's last CTA group) against a one-shot oracle run
    at full nt (the oracle uses its own stride-100 checkpointing: its full history would be 105 GB)."""
    wl = gi.config4()
    budget = _bench_budget()
    p = params_of(wl)
    _, plan0 = gprfwi_workspace_bytes(p, budget)
    assert plan0["full_history"] == 0 and 1 < plan0["shots_per_pass"] < wl.nshots
    plan = _one_hot_residual_case(wl, plan0["shots_per_pass"] - 1, budget, oracle_stride=100)
    assert plan == plan0


def test_config5_512_full_nt_and_1024_batch32_against_oracle():
    """Config 5 at its full nt = 1000: 512^2 with B = 8 (shots 0 and 7 against the oracle), and 1024^2 with
    B = 32 in one call (one-hot residual on shot 31)."""
    wl = gi.config5(n=512, batch=8)
    sub = wl.subset([0, 7])
    tr_o, res_sub, ge_o, gs_o = oracle_all(sub)
    res = np.zeros((wl.nshots, wl.nt, wl.nrec), dtype=np.float32)
    res[[0, 7]] = res_sub
    tr, ge, gs, plan = run_gpu(wl, res)
    assert plan["shots_per_pass"] == 8
    # SURVEY's recipe for config 5 is a WHITE-NOISE residual: injected at a receiver 11 cells from a source of
    # this strongly lossy i.i.d. medium it leaves single receiver cells 4e-4 of the peak off (the fp32
    # wavefield, not the accumulation: runs with 2 and 4 fused steps agree to 3e-7 there, and the physical
    # residual below is exact to 1e-6), so the whole-array bar holds and the local ones are 1e-3 here ...
    assert_parity(sub, (tr[[0, 7]], ge, gs), (tr_o, ge_o, gs_o), " 512^2 B=8 full nt, white-noise residual",
                  tol_region=1e-3, tol_maxabs=1e-3)
    # ... and strict with a band-limited residual (the shots' own traces)
    res[[0, 7]] = tr_o.astype(np.float32)
    ge_o2, gs_o2 = oracle.gradient(problem(sub), sub.eps_r, sub.sigma, res[[0, 7]])
    _, ge2, gs2, _ = run_gpu(wl, res)
    assert_parity(sub, (tr[[0, 7]], ge2, gs2), (tr_o, ge_o2, gs_o2), " 512^2 B=8 full nt, residual = traces")
    _one_hot_residual_case(gi.config5(n=1024, batch=32), 31, _bench_budget(), oracle_stride=0, tol_local=1e-3)


def test_config5_8192_grid_short_run_and_batch128_against_oracle():
    """The two corners of config 5's sweep that bench.py times and no other test touches: the 8192 x 8192 grid
    (20 520 tiles, plane offsets beyond 2^26 cells) for 16 steps with one source near the bottom-right corner and
    six receivers within reach of the wave -- everything the wave has not reached must stay exactly zero --, and
    512^2 with B = 128 shots in ONE call at the full nt = 1000 (one-hot residual on the last shot)."""
    import dataclasses
    wl = gi.config5(n=8192, batch=1, nt=16)
    off = np.array([(2, 0), (0, 3), (-3, -1), (4, 4), (-2, 2), (1, -4)])
    src = np.array([(8150, 8160)])
    wl = gi.with_geometry(wl, src, src[:, None, :] + off[None, :, :], name="config5-8192-short")
    wl = dataclasses.replace(wl, wavelet=np.sin(0.6 * np.arange(16)).astype(np.float32))
    pb = problem(wl)
    tr_o = oracle.forward(pb, wl.eps_r, wl.sigma)["traces"]
    res = gi.random_residual(wl, float(np.sqrt(np.mean(tr_o ** 2))))
    ge_o, gs_o = oracle.gradient(pb, wl.eps_r, wl.sigma, res, checkpoint_stride=4)      # (5 planes of 0.5 GB, not 17)
    tr, ge, gs, plan = run_gpu(wl, res)
    assert_parity(wl, (tr, ge, gs), (tr_o, ge_o, gs_o), " 8192^2, 16 steps")
    far = np.ones((wl.nz, wl.nx), bool)
    far[8150 - 40:8150 + 41, 8160 - 40:] = False
    assert np.all(ge[far] == 0.0) and np.all(gs[far] == 0.0) and np.all(ge_o[far] == 0.0)
    del tr, ge, gs, ge_o, gs_o, far
    plan = _one_hot_residual_case(gi.config5(n=512, batch=128), 127, _bench_budget(), oracle_stride=0, tol_local=1e-3)
    assert plan["shots_per_pass"] == 128 and plan["full_history"] == 1


def test_iteration_is_cuda_graph_capturable_after_one_warm_call():
    """The boundary's "calls only enqueue" contract, checked the hard way: after one warm call on a handle (which
    allocates the handle's pinned staging block and streams), forward -> residual -> adjoint on the same handle
    is captured into a CUDA graph -- programmatic dependent launches, the forked launch lanes and the memsets
    included -- and the replay, after the models were changed IN PLACE, is bit-identical to an eager run."""
    wl = gi.small_random(nz=70, nx=150, nt=60, npml=10, nshots=3, nrec=6, seed=515)
    sim = Simulation(params_of(wl), wl.src_zx, wl.rec_zx, wl.wavelet, dev())
    eps = torch.as_tensor(wl.eps_r.copy(), device=dev()); sig = torch.as_tensor(wl.sigma.copy(), device=dev())
    d_obs = torch.as_tensor(gi.random_residual(wl, 1.0), device=dev()); res = torch.empty_like(d_obs)

    def iteration():
        gprfwi_residual(sim.forward(eps, sig), d_obs, res)
        sim.adjoint(res)

    side = torch.cuda.Stream()
    side.wait_stream(torch.cuda.current_stream())
    graph = torch.cuda.CUDAGraph()
    with torch.cuda.stream(side):
        iteration()                                    # warm call: everything that allocates happens here
        torch.cuda.synchronize()
        with torch.cuda.graph(graph, stream=side):
            iteration()
    torch.cuda.synchronize()
    eps.mul_(1.1); sig.add_(1e-3)                      # new models, same buffers
    for t in (sim.traces, sim.grad_eps_r, sim.grad_sigma):
        t.fill_(float("nan"))
    graph.replay()
    torch.cuda.synchronize()
    got = [t.clone() for t in (sim.traces, sim.grad_eps_r, sim.grad_sigma)]
    iteration()
    torch.cuda.synchronize()
    for a, b in zip(got, (sim.traces, sim.grad_eps_r, sim.grad_sigma)):
        assert torch.isfinite(a).all() and torch.equal(a, b)
    sim.close()


def test_split_batch_multi_call_sum_against_oracle():
    """bench.py sweeps a batch that does not fit one call as several calls through one workspace and sums the
    gradients (split_batch picks the split): 512^2, B = 8, nt = 400 under a budget that forces more than
    one call, summed as bench.py sums it, against the oracle's gradient of all 8 shots."""
    from paper_2506_20513_b200 import split_batch
    wl = gi.config5(n=512, batch=8, nt=400)
    p = params_of(wl)
    lo, hi = 1 << 20, gprfwi_workspace_bytes(p, 0)[0]               # smallest workspace the 8 shots fit in one call
    while hi - lo > (1 << 16):
        mid = (lo + hi) // 2
        lo, hi = (lo, mid) if gprfwi_workspace_bytes(p, mid)[0] else (mid, hi)
    budget = lo                                                     # ... and just below it: the batch must be split
    assert gprfwi_workspace_bytes(p, budget)[0] == 0
    ncalls, cs, plan = split_batch(p, budget)
    print("[split]", ncalls, "calls of", cs, "shots:", plan)
    assert ncalls > 1 and ncalls * cs == wl.nshots
    tr_o, res, ge_o, gs_o = oracle_all(wl)
    p.nshots = cs
    sim = Simulation(p, wl.src_zx[:cs], wl.rec_zx[:cs], wl.wavelet, dev(), budget_bytes=budget)
    e = torch.as_tensor(wl.eps_r, device=dev()); s_ = torch.as_tensor(wl.sigma, device=dev())
    ge = torch.zeros_like(e); gs = torch.zeros_like(e)
    tr = np.zeros_like(tr_o, dtype=np.float32)
    for ci in range(ncalls):
        sl = slice(ci * cs, (ci + 1) * cs)
        sim.src_zx, sim.rec_zx = wl.src_zx[sl], wl.rec_zx[sl]
        tr[sl] = sim.forward(e, s_).cpu().numpy()
        a, b = sim.adjoint(torch.as_tensor(res[sl], device=dev()))
        ge += a; gs += b
    sim.close()
    assert_parity(wl, (tr, ge.cpu().numpy(), gs.cpu().numpy()), (tr_o, ge_o, gs_o), f" {ncalls} calls of {cs} shots",
                  tol_region=1e-3, tol_maxabs=1e-3)           # (white-noise residual on config 5: see above)


def test_mu_r_model_against_oracle_and_unit_permeability_bit_identical():
    """SURVEY 8(f)-3, reading R22: a heterogeneous relative permeability (Table 1 `miu`) through
    gprfwi_forward_mu against the oracle (ragged grid, CPML, several tiles, stored history and
    checkpoint-and-recompute), and mu_r = 1 everywhere bit-identical to the call without a mu_r model."""
    wl = gi.small_random(nz=97, nx=263, nt=180, npml=12, nshots=3, nrec=7, seed=97263)
    rng = np.random.default_rng(11)
    mu = rng.uniform(1.0, 3.0, (wl.nz, wl.nx)).astype(np.float32)
    pb = problem(wl)
    tr_o = oracle.forward(pb, wl.eps_r, wl.sigma, mu_r=mu)["traces"]
    res = gi.random_residual(wl, float(np.sqrt(np.mean(tr_o ** 2))))
    ge_o, gs_o = oracle.gradient(pb, wl.eps_r, wl.sigma, res, mu_r=mu)
    assert rel_l2(tr_o, oracle.forward(pb, wl.eps_r, wl.sigma)["traces"]) > 1e-2        # mu_r matters here
    pitch = wl.nx + 5
    e = torch.as_tensor(padded(wl.eps_r, pitch), device=dev()); s_ = torch.as_tensor(padded(wl.sigma, pitch), device=dev())
    ones = torch.ones((wl.nz, pitch), device=dev())
    m = torch.as_tensor(padded(mu, pitch), device=dev()); m[:, wl.nx:] = 1.0
    out = {}
    for K in (0, 16):
        sim = Simulation(params_of(wl, pitch=pitch, checkpoint_stride=K), wl.src_zx, wl.rec_zx, wl.wavelet, dev())
        sim.workspace.fill_(0xFF)
        for tag, model in (("none", None), ("ones", ones), ("mu", m)):
            tr = sim.forward(e, s_, mu_r=model).cpu().numpy().copy()
            a, b = sim.adjoint(torch.as_tensor(res, device=dev()))
            out[tag, K] = (tr, a.cpu().numpy()[:, :wl.nx].copy(), b.cpu().numpy()[:, :wl.nx].copy())
        sim.close()
        for x, y in zip(out["none", K], out["ones", K]):
            assert np.array_equal(x, y)
        assert_parity(wl, out["mu", K], (tr_o, ge_o, gs_o), f" mu_r model, K = {K}")
    assert np.array_equal(out["mu", 0][0], out["mu", 16][0])


def test_grid_transfer_kernels_and_coarse_stage():
    """SURVEY 8(f)-2 remainder (reading R23): gprfwi_restrict / gprfwi_prolong_add against the
    NumPy oracle on odd and even grids with a row pitch, and a coarse-grid stage of invert_staged: its first
    misfit equals the oracle's misfit of the COARSE problem (restricted models, doubled dx, halved CPML,
    geometry on the nearest coarse nodes, low-passed wavelet and data), the fine models move by the
    prolongation of the coarse update, and the stage lowers its misfit."""
    from oracle import epilogue as ep
    from paper_2506_20513_b200 import (Stage, invert_staged, coarse_problem, gprfwi_restrict, gprfwi_prolong_add)
    rng = np.random.default_rng(31)
    for nz, nx in ((41, 57), (40, 130), (97, 263)):
        f = rng.standard_normal((nz, nx)).astype(np.float32)
        d_f = torch.zeros((nz, nx + 3), device=dev()); d_f[:, :nx] = torch.as_tensor(f, device=dev())
        d_c = gprfwi_restrict(d_f[:, :nx])
        assert rel_l2(d_c.cpu().numpy(), ep.restrict(f)) <= 1e-6
        base = rng.standard_normal((nz, nx)).astype(np.float32)
        d_b = torch.as_tensor(base.copy(), device=dev())
        gprfwi_prolong_add(d_c, d_b, scale=-0.5)
        assert rel_l2(d_b.cpu().numpy(), base - 0.5 * ep.prolong(d_c.cpu().numpy(), nz, nx)) <= 1e-6
        assert torch.all(d_f[:, nx:] == 0)
    wl = gi.crosshole(nt=600)
    pb = problem(wl)
    d_obs64 = oracle.forward(pb, wl.eps_r_obs, wl.sigma_obs)["traces"]
    d_obs = torch.as_tensor(d_obs64.astype(np.float32), device=dev())
    sim = Simulation(params_of(wl), wl.src_zx, wl.rec_zx, wl.wavelet, dev())
    eps = torch.as_tensor(wl.eps_r.copy(), device=dev()); sig = torch.as_tensor(wl.sigma.copy(), device=dev())
    hist = invert_staged(sim, eps, sig, d_obs, [Stage(4, 0.05, 0.0, f_cut=60e6, coarsen=True)], mask_rows=0,
                         tv_iters=3, tv_lambda=0.002, tv_alpha=0.0)
    pc, src_c, rec_c = coarse_problem(sim.p, wl.src_zx, wl.rec_zx)
    sim.close()
    print("[coarse stage]", " ".join(f"{h:.3e}" for h in hist[0]))
    assert (pc.nz, pc.nx, pc.npml) == ((wl.nz + 1) // 2, (wl.nx + 1) // 2, (wl.npml + 1) // 2)
    taps = ep.lowpass_design(wl.dt, 60e6)
    w_lp = ep.lowpass(wl.wavelet[None, :, None], taps)[0, :, 0]
    d_lp = ep.lowpass(d_obs.cpu().numpy(), taps)
    pbc = oracle.Problem(nz=pc.nz, nx=pc.nx, dx=2.0 * wl.dx, dt=wl.dt, nt=wl.nt, npml=pc.npml, pml_order=wl.pml_order,
                         pml_sigma_max=0.5 * wl.pml_sigma_max, pml_kappa_max=wl.pml_kappa_max,
                         pml_alpha_max=wl.pml_alpha_max, src_zx=src_c, rec_zx=rec_c, wavelet=w_lp)
    r0 = oracle.forward(pbc, ep.restrict(wl.eps_r), ep.restrict(wl.sigma))["traces"] - d_lp
    assert abs(hist[0][0] - 0.5 * np.sum(r0 * r0)) <= 1e-3 * hist[0][0]
    assert hist[0][-1] < hist[0][0]
    de = eps.cpu().numpy() - wl.eps_r
    assert np.abs(de).max() > 0 and torch.equal(sig.cpu(), torch.as_tensor(wl.sigma))      # lr_sigma = 0
    # the update is a bilinear field: it is reproduced by prolonging its own values at the even nodes
    assert rel_l2(ep.prolong(de[::2, ::2], wl.nz, wl.nx), de) <= 1e-5
