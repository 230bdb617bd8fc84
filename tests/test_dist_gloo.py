"""N > 1 host path on CPU: world_size-2 gloo.  Each rank takes its shard of the shots, computes that
shard's gradient (with the oracle standing in for the GPU sweep -- this test is about the sharding
and the reduction, not the kernels) and the all-reduced sum must equal the full-batch gradient."""
import os
import socket

import numpy as np
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
