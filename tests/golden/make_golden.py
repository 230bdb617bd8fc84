"""Writes tests/golden/config1_oracle.txt from the float64 oracle ONLY (never from the CUDA path).

The paper (arxiv/paper_2506_20513) prints no trace, gradient or loss value, so
there is no paper-given worked example to store; this file freezes a handful of oracle numbers of
BASELINE.json config 1 so that an accidental change to the oracle's arithmetic (or to the input
generator) is noticed.  Run from the repo root:  python tests/golden/make_golden.py
"""
import os
import sys

import numpy as np

ROOT = os.path.dirname(os.path.dirname(os.path.dirname(os.path.abspath(__file__))))
sys.path.insert(0, ROOT)
sys.path.insert(0, os.path.join(ROOT, "tests"))

import gpr_inputs as gi  # noqa: E402
import oracle  # noqa: E402
from helpers import problem  # noqa: E402


def values():
    oracle.build()
    wl = gi.config1()
    pb = problem(wl)
    tr = oracle.forward(pb, wl.eps_r, wl.sigma)["traces"]
    obs = oracle.forward(pb, wl.eps_r_obs, wl.sigma_obs)["traces"]
    res = (tr - obs).astype(np.float32)
    ge, gs = oracle.gradient(pb, wl.eps_r, wl.sigma, res)
    out = {"misfit": 0.5 * float(np.sum(res.astype(np.float64) ** 2)),
           "trace_l2": float(np.linalg.norm(tr)), "grad_eps_r_l2": float(np.linalg.norm(ge)),
           "grad_sigma_l2": float(np.linalg.norm(gs))}
    for n in (200, 400, 600, 799):
        for r in (0, 4, 9):
            out[f"trace[0][{n}][{r}]"] = float(tr[0, n, r])
    for (j, i) in ((15, 60), (60, 60), (80, 40)):
        out[f"grad_eps_r[{j}][{i}]"] = float(ge[j, i])
        out[f"grad_sigma[{j}][{i}]"] = float(gs[j, i])
    return out


if __name__ == "__main__":
    path = os.path.join(os.path.dirname(os.path.abspath(__file__)), "config1_oracle.txt")
    with open(path, "w") as f:
        f.write("# BASELINE.json config 1, float64 oracle (oracle/gprfwi_oracle.c); written by make_golden.py\n")
        for k, v in values().items():
            f.write(f"{k} {v:.15e}\n")
    print("wrote", path)
