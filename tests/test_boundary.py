"""CPU-side checks of the C-ABI boundary: the library loads, exports every symbol include/gprfwi.h
declares, validates arguments and plans memory.  No compute calls (no GPU here)."""
import ctypes
import os
import re

import numpy as np
import pytest

import gpr_inputs as gi
from paper_2506_20513_b200 import _lib, build, make_params, gprfwi_workspace_bytes, gprfwi_workspace_bytes_host

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def lib():
    build.build()
    return _lib.load()


def params_of(wl, **over):
    kw = dict(nz=wl.nz, nx=wl.nx, dx=wl.dx, dt=wl.dt, nt=wl.nt, npml=wl.npml, pml_order=wl.pml_order,
              pml_sigma_max=wl.pml_sigma_max, pml_kappa_max=wl.pml_kappa_max, pml_alpha_max=wl.pml_alpha_max,
              nshots=wl.nshots, nrec=wl.nrec)
    kw.update(over)
    return make_params(**kw)


def test_every_declared_symbol_is_exported(lib):
    text = open(os.path.join(ROOT, "include", "gprfwi.h")).read()
    text = re.sub(r"/\*.*?\*/", "", text, flags=re.S)
    declared = set(re.findall(r"\b(gprfwi_[a-z_]+)\s*\(", text))
    assert declared == set(_lib.EXPORTS), declared ^ set(_lib.EXPORTS)
    for name in declared:
        assert hasattr(lib, name), name
    assert lib.gprfwi_version() >= 100


def test_struct_layout_matches_header():
    assert ctypes.sizeof(_lib.Params) == 15 * 4
    assert ctypes.sizeof(_lib.Plan) == 8 + 6 * 4


def test_strerror(lib):
    for code in range(0, -7, -1):
        assert len(lib.gprfwi_strerror(code)) > 0


def test_invalid_params_give_zero_workspace(lib):
    wl = gi.config1(nt=10)
    assert gprfwi_workspace_bytes(params_of(wl))[0] > 0
    assert gprfwi_workspace_bytes(params_of(wl, nt=0))[0] == 0
    assert gprfwi_workspace_bytes(params_of(wl, pitch=wl.nx - 1))[0] == 0
    assert gprfwi_workspace_bytes(params_of(wl, nz=2 * wl.npml + 2))[0] == 0
    assert gprfwi_workspace_bytes(params_of(wl, dx=0.0))[0] == 0
    assert gprfwi_workspace_bytes(params_of(wl, dt=wl.dx / (gi.C0 * np.sqrt(2)) * 1.01))[0] == 0   # CFL, Eq. (11)


def test_forward_rejects_bad_arguments_before_touching_the_gpu(lib):
    wl = gi.config1(nt=10)
    h = ctypes.c_void_p(None)
    p = params_of(wl, dt=1e-9)
    one = ctypes.c_void_p(256)
    rc = lib.gprfwi_forward(ctypes.byref(h), ctypes.byref(p), one, one, one, one, one, one, 1 << 30, one, None)
    assert rc == -2                                   # ECFL
    p = params_of(wl)
    rc = lib.gprfwi_forward(ctypes.byref(h), ctypes.byref(p), None, one, one, one, one, one, 1 << 30, one, None)
    assert rc == -1                                   # EINVAL: null model
    rc = lib.gprfwi_forward(ctypes.byref(h), ctypes.byref(p), one, one, one, one, one, one, 1024, one, None)
    assert rc == -4                                   # ENOMEM: workspace too small
    assert lib.gprfwi_adjoint(None, one, one, one, None) == -1


def test_plan_full_history_when_it_fits_else_checkpoints(lib):
    wl = gi.config2(nt=3000)
    p = params_of(wl)
    nb, plan = gprfwi_workspace_bytes(p, 0)
    assert plan["full_history"] == 1 and plan["shots_per_pass"] == 20
    hist = (wl.nt + 1) * wl.nshots * wl.nz * 448 * 4      # pitch 440 -> 448
    assert hist <= nb <= hist * 1.02
    nb2, plan2 = gprfwi_workspace_bytes(p, nb // 4)
    assert 0 < nb2 <= nb // 4 and plan2["full_history"] == 0 and 1 < plan2["checkpoint_stride"] < wl.nt
    # config 3 and 4 need recompute inside 170 GB; config 4 also needs shot sub-batches
    budget = 170 * 10 ** 9
    p3 = make_params(nz=540, nx=1040, dx=0.01, dt=2e-11, nt=4000, npml=20, pml_order=3, pml_sigma_max=1.0,
                     pml_kappa_max=1.0, pml_alpha_max=0.0, nshots=60, nrec=200)
    nb3, plan3 = gprfwi_workspace_bytes(p3, budget)
    assert 0 < nb3 <= budget and plan3["full_history"] == 0 and plan3["shots_per_pass"] == 60
    # spare budget holds the Ez planes of the last segments; none of it when the budget is the bare minimum
    nseg3 = -(-p3.nt // plan3["checkpoint_stride"])
    assert 0 < plan3["stored_segments"] < nseg3
    per3 = (plan3["checkpoint_stride"] - 1) * 60 * 540 * 1056 * 4
    bare = nb3 - plan3["stored_segments"] * per3
    nb3b, plan3b = gprfwi_workspace_bytes(p3, bare + 1024)
    assert plan3b["stored_segments"] == 0 and plan3b["checkpoint_stride"] == plan3["checkpoint_stride"]
    assert abs(nb3b - bare) < 4096
    p4 = make_params(nz=1060, nx=2060, dx=0.005, dt=1e-11, nt=6000, npml=30, pml_order=3, pml_sigma_max=1.0,
                     pml_kappa_max=1.0, pml_alpha_max=0.0, nshots=100, nrec=400)
    nb4, plan4 = gprfwi_workspace_bytes(p4, budget)
    assert 0 < nb4 <= budget and plan4["full_history"] == 0 and plan4["shots_per_pass"] < 100
    assert gprfwi_workspace_bytes(p4, 10 ** 9)[0] == 0      # nothing fits in 1 GB
    assert gprfwi_workspace_bytes_host(p, 0) > nb


def test_forced_stride(lib):
    wl = gi.config1(nt=100)
    nb, plan = gprfwi_workspace_bytes(params_of(wl, checkpoint_stride=7), 0)
    assert plan["full_history"] == 0 and plan["checkpoint_stride"] == 7


def test_acquisition_presets_match_table_1_semantics():
    """step / source_step / receiver_step / Fixedreceiver as integer-cell positions."""
    import gpr_inputs as gi
    src, rec = gi.acquisition((15, 20), (0, 4), 5, (15, 22), (0, 1), 3)
    assert src.tolist() == [[15, 20 + 4 * k] for k in range(5)]
    assert rec[:, :, 1].tolist() == [[22 + 4 * k + j for j in range(3)] for k in range(5)]      # array moves along
    assert np.all(rec[:, :, 0] == 15)
    _, rec_f = gi.acquisition((15, 20), (0, 4), 5, (15, 22), (0, 1), 3, fixed_receiver=True)
    assert np.all(rec_f == rec[:1])
    wl = gi.crosshole()
    assert (wl.nz, wl.nx, wl.nshots, wl.nrec, wl.nt) == (220, 120, 1, 200, 1000)
    assert np.all(np.diff(wl.rec_zx[0, :, 0]) == 1) and np.all(wl.rec_zx[0, :, 1] == wl.rec_zx[0, 0, 1])
    with pytest.raises(AssertionError):
        gi.with_geometry(wl, [[0, 5]], [[[5, 5]]])                                          # on the PEC ring


def test_split_batch_prefers_plans_with_several_shots_per_pass():
    """Host-side planning only: a batch that fits one call only with single-shot adjoint passes is split."""
    from paper_2506_20513_b200 import split_batch
    mk = lambda n, b: make_params(nz=n, nx=n, dx=0.01, dt=2e-11, nt=1000, npml=10, pml_order=3, pml_sigma_max=1.0,
                                  pml_kappa_max=1.0, pml_alpha_max=0.1, nshots=b, nrec=64)
    budget = int(165e9)
    p = mk(4096, 128)
    nbytes, plan1 = gprfwi_workspace_bytes(p, budget)
    assert nbytes == 0 or plan1["shots_per_pass"] < 3                     # one call: does not fit, or barely
    ncalls, per_call, plan = split_batch(p, budget)
    assert ncalls * per_call == 128 and ncalls > 1 and plan["shots_per_pass"] >= 3
    assert p.nshots == 128                                                # params restored
    assert split_batch(mk(512, 8), budget)[:2] == (1, 8)                  # fits with full history: no split
    with pytest.raises(ValueError):
        split_batch(mk(8192, 4), int(1e9))                                # one shot does not fit 1 GB


def test_lowpass_design_host_call_matches_oracle():
    """gprfwi_lowpass_design runs on the host (no GPU needed): its taps against the oracle's NumPy statement
    (itself pinned against scipy.signal.firwin), the size query, and the error returns."""
    import numpy as np
    from oracle import epilogue as ep
    lib = _lib.load()
    for dt, f_cut, ntaps in ((2e-11, 150e6, 0), (1e-10, 80e6, 0), (2e-11, 400e6, 33)):
        n = lib.gprfwi_lowpass_design(dt, f_cut, ntaps, None)
        ref = ep.lowpass_design(np.float32(dt), np.float32(f_cut), ntaps)
        assert n == len(ref)
        taps = np.zeros(n, dtype=np.float32)
        assert lib.gprfwi_lowpass_design(dt, f_cut, ntaps, taps.ctypes.data) == n
        assert np.allclose(taps, ref, rtol=2e-7, atol=1e-9)
    assert lib.gprfwi_lowpass_design(2e-11, 150e6, 32, None) == -1            # even tap count
    assert lib.gprfwi_lowpass_design(0.0, 150e6, 0, None) == -1
