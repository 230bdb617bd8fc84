"""gprfwi_update_noalloc: the iteration epilogue with its TV scratch in the library's fixed device array
(no workspace argument, no allocation) against the existing gprfwi_update path.  Collected last on purpose
(the suite runs with pytest -x): it must pass alone in a fresh process and after all other tests."""
import numpy as np
import pytest
import torch

import gpr_inputs as gi
from helpers import rel_l2
from paper_2506_20513_b200 import (GprfwiError, gprfwi_update, gprfwi_update_noalloc, gprfwi_update_noalloc_max_bytes,
                                   gprfwi_update_workspace_bytes, make_update_params)

pytestmark = pytest.mark.gpu

TOL = 1e-5          # what test_epilogue_update_matches_numpy_oracle asserts on the updated models


def _planes(a, pitch, dev):
    out = torch.zeros((a.shape[0], pitch), device=dev)
    out[:, :a.shape[1]] = torch.as_tensor(a.astype(np.float32), device=dev)
    return out


def test_update_noalloc_matches_workspace_path_on_two_calls_in_a_row():
    assert torch.cuda.is_available(), "this test needs a CUDA device"
    dev = torch.device("cuda:0")
    assert gprfwi_update_noalloc_max_bytes() == 7 * (1 << 20) * 4 + 256
    rng = np.random.default_rng(19)
    # two different problems back to back: the second call meets the first one's leftovers in the shared scratch
    for call, (nz, nx, pad) in enumerate(((70, 150, 3), (240, 440, 0))):
        wl = gi.small_random(nz=nz, nx=nx, nt=10, npml=10, nshots=1, nrec=2, seed=50 + call)
        pitch = nx + pad
        assert gprfwi_update_workspace_bytes(nz, pitch) <= gprfwi_update_noalloc_max_bytes()
        ws = torch.empty(gprfwi_update_workspace_bytes(nz, pitch), dtype=torch.uint8, device=dev)
        ws.fill_(0xFF)
        state = {}
        for path in ("workspace", "noalloc"):
            eps, sig = _planes(wl.eps_r, pitch, dev), _planes(wl.sigma, pitch, dev)
            mom = [torch.zeros((nz, pitch), device=dev) for _ in range(4)]
            state[path] = (eps, sig, mom, [])
        for step in (1, 2):
            ge = rng.standard_normal((nz, nx)) * 1e-3
            gs = rng.standard_normal((nz, nx)) * 2.0
            u = make_update_params(step=step, lr_eps_r=0.05, lr_sigma=2e-4, tv_iters=10, tv_lambda=0.01,
                                   mask_rows=16, eps_r_min=1.0, sigma_min=0.0)
            for path, (eps, sig, mom, grads) in state.items():
                d_ge, d_gs = _planes(ge, pitch, dev), _planes(gs, pitch, dev)
                if path == "workspace":
                    gprfwi_update(nz, nx, pitch, u, eps, sig, d_ge, d_gs, mom[0], mom[1], mom[2], mom[3], ws)
                else:
                    gprfwi_update_noalloc(nz, nx, pitch, u, eps, sig, d_ge, d_gs, mom[0], mom[1], mom[2], mom[3])
                grads[:] = [d_ge, d_gs]
            torch.cuda.synchronize()
            a, b = state["workspace"], state["noalloc"]
            for name, x, y in (("eps_r", a[0], b[0]), ("sigma", a[1], b[1]), ("grad_eps_r+tv", a[3][0], b[3][0]),
                               ("grad_sigma+tv", a[3][1], b[3][1]), ("m_eps_r", a[2][0], b[2][0]),
                               ("v_sigma", a[2][3], b[2][3])):
                err = rel_l2(y.cpu().numpy(), x.cpu().numpy())
                assert err <= TOL, (call, step, name, err)
            assert not torch.equal(a[0][:, :nx], _planes(wl.eps_r, pitch, dev)[:, :nx])       # the step did move the model
            assert torch.all(b[0][:, nx:] == 0)                                              # pitch padding untouched


def test_update_noalloc_rejects_models_beyond_the_fixed_scratch():
    dev = torch.device("cuda:0")
    nz, nx = 1100, 1100                                  # 1.21 M cells > 2^20
    assert gprfwi_update_workspace_bytes(nz, nx) > gprfwi_update_noalloc_max_bytes()
    t = [torch.ones((nz, nx), device=dev) for _ in range(8)]
    before = t[0].clone()
    u = make_update_params(step=1, lr_eps_r=0.05, lr_sigma=2e-4)
    with pytest.raises(GprfwiError) as ei:
        gprfwi_update_noalloc(nz, nx, nx, u, *t)
    assert ei.value.code == -7 and "gprfwi_update_noalloc" in str(ei.value)
    torch.cuda.synchronize()
    assert torch.equal(t[0], before)                     # nothing was enqueued
