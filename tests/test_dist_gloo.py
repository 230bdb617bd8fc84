"""N > 1 host path on CPU: world_size-2 gloo.  Each rank takes its shard of the shots, computes that
shard's gradient (with the oracle standing in for the GPU sweep -- this test is about the sharding
and the reduction, not the kernels) and the all-reduced sum must equal the full-batch gradient."""
import os
import socket

import numpy as np
import pytest
import torch
import torch.distributed as dist
import torch.multiprocessing as mp

import gpr_inputs as gi
import oracle
from helpers import problem
from paper_2506_20513_b200.dist import allreduce_gradients, shard_shots


def test_shard_shots_partitions():
    for n in (1, 5, 20, 61):
        for w in (1, 2, 3, 8):
            got = [i for r in range(w) for i in shard_shots(n, r, w)]
            assert got == list(range(n))
            sizes = [len(shard_shots(n, r, w)) for r in range(w)]
            assert max(sizes) - min(sizes) <= 1


def _worker(rank, world, port, out):
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    wl = gi.small_random(nz=40, nx=46, nt=60, npml=6, nshots=5, nrec=4, seed=3)
    res = gi.random_residual(wl, 1.0, seed=11)
    mine = list(shard_shots(wl.nshots, rank, world))
    sub = wl.subset(mine)
    ge, gs = oracle.gradient(problem(sub), sub.eps_r, sub.sigma, res[mine])
    ge, gs = torch.from_numpy(np.ascontiguousarray(ge)), torch.from_numpy(np.ascontiguousarray(gs))
    allreduce_gradients(ge, gs)
    if rank == 0:
        np.save(out, np.stack([ge.numpy(), gs.numpy()]))
    dist.destroy_process_group()


def test_sharded_gradients_allreduce_to_full_batch(tmp_path):
    oracle.build()
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0)); port = s.getsockname()[1]
    out = str(tmp_path / "g.npy")
    mp.spawn(_worker, args=(2, port, out), nprocs=2, join=True)
    got = np.load(out)
    wl = gi.small_random(nz=40, nx=46, nt=60, npml=6, nshots=5, nrec=4, seed=3)
    res = gi.random_residual(wl, 1.0, seed=11)
    ge, gs = oracle.gradient(problem(wl), wl.eps_r, wl.sigma, res)
    assert np.allclose(got[0], ge, rtol=1e-12, atol=1e-12 * np.abs(ge).max())
    assert np.allclose(got[1], gs, rtol=1e-12, atol=1e-12 * np.abs(gs).max())


def _gpu_worker(rank, world, port, out):
    """The real sweep (Simulation -> libgprfwi) on this rank's shard of the shots; the two ranks share one
    GPU but never wait on one another's kernels: each finishes its own sweep, then the two gradient planes
    are summed with one all-reduce (gloo here, NCCL over NVLink in bench.py --gpus N)."""
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    from paper_2506_20513_b200 import Simulation
    from test_boundary import params_of
    dev = torch.device("cuda:0")
    wl = gi.small_random(nz=70, nx=150, nt=120, npml=10, nshots=5, nrec=6, seed=303)
    res = gi.random_residual(wl, 1.0, seed=12)
    mine = list(shard_shots(wl.nshots, rank, world))
    sub = wl.subset(mine)
    sim = Simulation(params_of(sub), sub.src_zx, sub.rec_zx, sub.wavelet, dev)
    sim.forward(torch.as_tensor(wl.eps_r, device=dev), torch.as_tensor(wl.sigma, device=dev))
    ge, gs = sim.adjoint(torch.as_tensor(res[mine], device=dev))
    ge, gs = ge.cpu(), gs.cpu()
    sim.close()
    allreduce_gradients(ge, gs)
    if rank == 0:
        np.save(out, np.stack([ge.numpy(), gs.numpy()]))
    dist.destroy_process_group()


@pytest.mark.gpu
def test_sharded_simulation_path_allreduces_to_full_batch(tmp_path):
    """SURVEY 8(e) on the CUDA path: shots sharded over two ranks, one all-reduce of the two gradient planes;
    the sum equals the one-process full-batch gradient (fp32 regrouping only) and the oracle's."""
    from paper_2506_20513_b200 import Simulation
    from test_boundary import params_of
    oracle.build()
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0)); port = s.getsockname()[1]
    out = str(tmp_path / "g.npy")
    mp.spawn(_gpu_worker, args=(2, port, out), nprocs=2, join=True)
    got = np.load(out)
    dev = torch.device("cuda:0")
    wl = gi.small_random(nz=70, nx=150, nt=120, npml=10, nshots=5, nrec=6, seed=303)
    res = gi.random_residual(wl, 1.0, seed=12)
    sim = Simulation(params_of(wl), wl.src_zx, wl.rec_zx, wl.wavelet, dev)
    sim.forward(torch.as_tensor(wl.eps_r, device=dev), torch.as_tensor(wl.sigma, device=dev))
    ge, gs = [t.cpu().numpy() for t in sim.adjoint(torch.as_tensor(res, device=dev))]
    sim.close()
    ge_o, gs_o = oracle.gradient(problem(wl), wl.eps_r, wl.sigma, res)
    for a, b, c in ((got[0], ge, ge_o), (got[1], gs, gs_o)):
        assert np.linalg.norm(a - b) <= 1e-5 * np.linalg.norm(b)
        assert np.linalg.norm(a - c) <= 1e-4 * np.linalg.norm(c)
