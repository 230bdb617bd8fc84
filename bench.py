#!/usr/bin/env python
"""bench.py -- forward+adjoint FDTD throughput of libgprfwi on BASELINE.json's configs.

A "step" is one FWI iteration = one pass of the whole hot path over one batch of synthetic input:
coefficient build, nt forward steps (H+E+CPML+source+receivers+history/checkpoints), residual + misfit,
nt adjoint steps with gradient accumulation (recompute sweeps included), chain rule, and the a7
epilogue (TV term, mask, Adam step, clamps).

Default workload: BASELINE.json configs[3] ("config4-high-frequency": 1060x2060 full grid, nt 6000,
100 shots, 400 receivers), the config the metric's "s per FWI iteration" is defined on and the largest
that fits one GPU; configs 2 and 3 are timed briefly in the same run and reported under `config.also`.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--config 1..5] [--impl ours|reference]

Prints ONE JSON line (rank 0).  `--gpus N` without torchrun re-executes itself under
`python -m torch.distributed.run --nproc-per-node N`; every rank then sweeps its own shard of
N x shots_per_gpu distinct shots (weak scaling) and one NCCL all-reduce sums the two gradient planes.
`--impl reference` times the float64 CPU oracle (oracle/) on a bounded sample instead.
"""
from __future__ import annotations

import argparse
import hashlib
import json
import os
import statistics
import subprocess
import sys
import threading
import time

import numpy as np

ROOT = os.path.dirname(os.path.abspath(__file__))
sys.path.insert(0, ROOT)
sys.path.insert(0, os.path.join(ROOT, "tests"))

import gpr_inputs as gi  # noqa: E402

METRIC = "forward+adjoint FDTD Gcell-updates/s"
UNIT = "Gcell-updates/s"
# algorithmic bytes per cell-step (SURVEY.md section 8(d), T = 1 figures)
BYTES_FWD, BYTES_ADJ, BYTES_RECOMPUTE = 28.0, 32.0, 28.0
DEFAULT_CONFIG = 4
ALSO = {4: (2, 3)}          # configs timed briefly beside the default one (north_star: configs 2 to 4)
TV_ITERS = 10


def load_workload(cfg: int, n: int = 512, batch: int = 1, world: int = 1):
    """The config's workload with `world` times its shots (distinct source positions on the same line)."""
    if cfg == 5:
        return gi.config5(n=n, batch=batch * world)
    if cfg == 1:
        wl = gi.config1()
        if world > 1:        # config 1 has one shot: replicate the line geometry with `world` sources
            src, rec = gi.line_geometry(wl.nz - 2 * wl.npml, wl.nx - 2 * wl.npml, wl.npml, world, wl.nrec)
            wl = gi.with_geometry(wl, src, rec, name=wl.name)
        return wl
    f = {2: gi.config2, 3: gi.config3, 4: gi.config4}[cfg]
    base = f()
    return base if world == 1 else f(nshots=base.nshots * world)


def peaks():
    path = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(path):
        with open(path) as f:
            return float(json.load(f)["hbm_gbs"]), "measured (MEASURED_PEAKS.json, burst copy)"
    return 6650.0, "fallback (B200_PROFILING.md)"


def kernel_source_sha() -> str:
    """Hash of the kernel sources (csrc/*.cuh): the key the ncu traffic table (profiles/dram_traffic.csv) is stored under
    (the GPU box has no .git, so a commit id cannot be read at run time)."""
    h = hashlib.sha256()
    d = os.path.join(ROOT, "paper_2506_20513_b200", "csrc")
    for f in sorted(os.listdir(d)):
        if f.endswith(".cuh"):            # the device code (kernels); host-only edits do not count
            with open(os.path.join(d, f), "rb") as fh:
                h.update(f.encode()); h.update(fh.read())
    return h.hexdigest()[:16]


def dram_traffic(cfg: int):
    """ncu-measured dram__bytes_read.sum + dram__bytes_write.sum per cell-step of each tile kernel on this
    config, from profiles/dram_traffic.csv (written by paper_2506_20513_b200/ncu_traffic.py from an
    `ncu --set full` capture; one row per config, build and part = fwd / recompute / adj).
    -> (dict(part -> bytes, "source" -> file) or None, stale flag): the rows of the build in the tree if the
    table has them, else the newest rows of another build, flagged stale."""
    import csv
    path = os.path.join(ROOT, "profiles", "dram_traffic.csv")
    if not os.path.exists(path):
        return None, None
    with open(path, newline="") as f:
        rows = [r for r in csv.DictReader(f) if int(r["config"]) == cfg]
    if not rows:
        return None, None
    sha = kernel_source_sha()
    mine = [r for r in rows if r["kernel_source_sha"] == sha]
    use = mine or [r for r in rows if r["kernel_source_sha"] == rows[-1]["kernel_source_sha"]]
    out = {r["part"]: float(r["dram_bytes_per_cell_step"]) for r in use}
    out["source"] = sorted({r["source"] for r in use})
    out["kernel_source_sha"] = use[-1]["kernel_source_sha"]
    return out, not mine


class ClockSampler:
    """nvidia-smi clocks / throttle reasons sampled during the timed region."""
    Q = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,"
         "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,"
         "clocks_event_reasons.sw_power_cap")

    def __init__(self, index: int):
        self.index, self.rows, self._stop, self._t = index, [], threading.Event(), None

    def _run(self):
        while not self._stop.is_set():
            try:
                out = subprocess.run(["nvidia-smi", f"--query-gpu={self.Q}", "--format=csv,noheader,nounits",
                                      "-i", str(self.index)], capture_output=True, text=True, timeout=5).stdout
                self.rows.append([c.strip() for c in out.strip().split(",")])
            except Exception:
                pass
            self._stop.wait(0.05)

    def __enter__(self):
        self._t = threading.Thread(target=self._run, daemon=True)
        self._t.start()
        return self

    def __exit__(self, *a):
        self._stop.set()
        self._t.join(timeout=6)

    def summary(self):
        sm, mx, reasons = [], [], set()
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        for r in self.rows:
            try:
                sm.append(float(r[0])); mx.append(float(r[1]))
                for k, nm in enumerate(names):
                    if r[3 + k].lower().startswith("active"):
                        reasons.add(nm)
            except Exception:
                continue
        return {"sm_mhz": statistics.median(sm) if sm else None, "sm_max_mhz": max(mx) if mx else None,
                "reasons": sorted(reasons), "samples": len(sm)}


# ------------------------------------------------------------------------------------------------
# the float64 CPU oracle, timed as it stands on a bounded sample (cpu_baseline leg / --impl reference)
# ------------------------------------------------------------------------------------------------
ORACLE_SAMPLE_CELL_UPDATES = 3.0e9          # per sample: about 10 s at the oracle's 0.3-0.45 Gcell-updates/s


def oracle_sample_shape(wl):
    """(number of shots, nt) of one bounded oracle sample of `wl`: whole shots at full nt while they fit
    the work bound, else one shot with the time axis cut (the per-step cost does not depend on nt)."""
    per_shot = 2.0 * wl.nz * wl.nx * wl.nt
    if per_shot <= ORACLE_SAMPLE_CELL_UPDATES:
        return max(1, min(wl.nshots, int(ORACLE_SAMPLE_CELL_UPDATES // per_shot))), wl.nt
    nt = int(ORACLE_SAMPLE_CELL_UPDATES / (2.0 * wl.nz * wl.nx))
    return 1, max(50, nt // 50 * 50)


def oracle_sample(wl, shots, nt):
    """Oracle forward+adjoint on some shots of the workload; returns (seconds, cell_updates)."""
    import oracle
    from helpers import problem
    sub = wl.subset(shots, nt=nt)
    res = gi.random_residual(sub, 1.0)
    t0 = time.perf_counter()
    oracle.gradient(problem(sub), sub.eps_r, sub.sigma, res)
    return time.perf_counter() - t0, sub.cell_updates


def run_reference(args, wl):
    """Reference arm of the bench contract for this tier: the oracle on the host cores, each step a bounded
    sample of the workload (different shots from step to step)."""
    import oracle
    oracle.build()
    ns, nt = oracle_sample_shape(wl)
    for _ in range(args.warmup):
        oracle_sample(wl, [0], min(nt, 100))
    times, work = [], 0
    for k in range(args.steps):
        shots = sorted({(k * 7 + j * max(1, wl.nshots // ns)) % wl.nshots for j in range(ns)})
        t, w = oracle_sample(wl, shots, nt)
        times.append(t); work += w
    total = sum(times)
    val = work / total / 1e9
    sample = (f"{args.steps} steps x {ns} shot(s) of {wl.name}, full grid, nt {nt} of {wl.nt}, float64, "
              f"OpenMP over rows")
    line = {"impl": "reference", "metric": METRIC, "value": val, "unit": UNIT, "n_gpus": args.gpus,
            "steps": args.steps, "warmup": args.warmup, "ms_per_step": 1e3 * total / args.steps,
            "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f64",
            "data": "synthetic", "config": {"workload": wl.name, "sample": sample},
            "cpu_baseline": {"value": val, "unit": UNIT, "cores": oracle.num_threads(), "kind": "oracle",
                             "sample": sample},
            "e2e": {"value": val, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
            "gpu_launches": 0}
    print(json.dumps(line))


# ------------------------------------------------------------------------------------------------
# the CUDA path
# ------------------------------------------------------------------------------------------------
def run_config(cfg, wl, steps, warmup, env, budget_gb=0.0, with_e2e=True, clocks_index=None):
    """Time `steps` FWI iterations of workload `wl` (this rank's shots) after `warmup` untimed ones.
    `env` = dict(dev, rank, world).  Returns a dict of measurements (times are max over ranks)."""
    import torch
    import torch.distributed as dist
    from paper_2506_20513_b200 import (Simulation, split_batch, gprfwi_gradient_host, gprfwi_residual,
                                       gprfwi_update, gprfwi_update_workspace_bytes, gprfwi_workspace_bytes_host,
                                       make_params, make_update_params)
    from paper_2506_20513_b200.dist import allreduce_gradients
    dev, world = env["dev"], env["world"]
    warmup = max(warmup, 3)

    p = make_params(nz=wl.nz, nx=wl.nx, dx=wl.dx, dt=wl.dt, nt=wl.nt, npml=wl.npml, pml_order=wl.pml_order,
                    pml_sigma_max=wl.pml_sigma_max, pml_kappa_max=wl.pml_kappa_max,
                    pml_alpha_max=wl.pml_alpha_max, nshots=wl.nshots, nrec=wl.nrec)
    torch.cuda.empty_cache()
    free, _total = torch.cuda.mem_get_info(dev)
    ntr = wl.nshots * wl.nt * wl.nrec
    budget = int(budget_gb * 1e9) if budget_gb > 0 else int(free * 0.92) - 3 * ntr * 4
    # A batch whose states do not fit one call, or fit only with single-shot adjoint passes (config 5's
    # largest cells), is split into equal chunks of shots that are swept one after the other through the
    # same workspace; gradients are summed (paper_2506_20513_b200.split_batch picks the split).
    try:
        nchunks, p.nshots, _ = split_batch(p, budget)
    except ValueError:
        raise SystemExit("the problem does not fit this GPU even one shot at a time")
    sim = Simulation(p, wl.src_zx[:p.nshots], wl.rec_zx[:p.nshots], wl.wavelet, dev, budget_bytes=budget)
    cs = p.nshots
    eps = torch.as_tensor(wl.eps_r, device=dev)
    sig = torch.as_tensor(wl.sigma, device=dev)
    # observed data: a seeded stand-in with the traces' scale (d_obs content does not change the work)
    rng = np.random.Generator(np.random.PCG64(wl.seed + 99 + env["rank"]))
    d_obs_h = (rng.standard_normal((wl.nshots, wl.nt, wl.nrec)) * 1e-3).astype(np.float32)
    d_obs = torch.as_tensor(d_obs_h, device=dev)
    res = torch.empty_like(d_obs)
    misfit = torch.zeros(1, dtype=torch.float64, device=dev)
    stream = torch.cuda.current_stream()
    # iteration epilogue (a7): TV term + mask + Adam + clamps on copies of the models, so that every
    # timed step runs the same forward problem (the step size is tiny and the copies are reset)
    eps_it, sig_it = eps.clone(), sig.clone()
    ge_acc, gs_acc = torch.zeros_like(eps), torch.zeros_like(eps)
    adam = [torch.zeros_like(eps) for _ in range(4)]
    ws_up = torch.empty(gprfwi_update_workspace_bytes(wl.nz, wl.nx), dtype=torch.uint8, device=dev)
    upd = make_update_params(step=1, lr_eps_r=1e-3, lr_sigma=1e-6, tv_iters=TV_ITERS, mask_rows=wl.npml + 7)

    def step(timers=None):
        ev = [torch.cuda.Event(enable_timing=True) for _ in range(5)] if timers is not None else None
        misfit.zero_()
        for ci in range(nchunks - 1):      # all chunks but the last (untimed split; the total time is what counts)
            sl = slice(ci * cs, (ci + 1) * cs)
            sim.src_zx, sim.rec_zx = wl.src_zx[sl], wl.rec_zx[sl]
            gprfwi_residual(sim.forward(eps, sig), d_obs[sl], res[sl], misfit)
            ge, gs = sim.adjoint(res[sl])
            if ci == 0: ge_acc.copy_(ge); gs_acc.copy_(gs)
            else: ge_acc.add_(ge); gs_acc.add_(gs)
        sl = slice((nchunks - 1) * cs, nchunks * cs)
        sim.src_zx, sim.rec_zx = wl.src_zx[sl], wl.rec_zx[sl]
        if ev: ev[0].record(stream)
        tr = sim.forward(eps, sig)
        if ev: ev[1].record(stream)
        gprfwi_residual(tr, d_obs[sl], res[sl], misfit)
        if ev: ev[2].record(stream)
        ge, gs = sim.adjoint(res[sl])
        if nchunks > 1: ge.add_(ge_acc); gs.add_(gs_acc)
        allreduce_gradients(ge, gs)        # shots are sharded over ranks: sum the gradients (no-op at N = 1)
        if ev: ev[3].record(stream)
        gprfwi_update(wl.nz, wl.nx, wl.nx, upd, eps_it, sig_it, ge, gs, adam[0], adam[1], adam[2], adam[3], ws_up)
        if ev:
            ev[4].record(stream)
            timers.append(ev)

    def barrier():
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    def max_over_ranks(x):
        if world > 1:
            t = torch.tensor([x], device=dev, dtype=torch.float64)
            dist.all_reduce(t, op=dist.ReduceOp.MAX)
            return float(t.item())
        return x

    for _ in range(warmup):
        step()
    barrier()
    timers = []
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)

    class _NoClocks:
        def __enter__(self): return self
        def __exit__(self, *a): pass
        def summary(self): return None

    with (ClockSampler(clocks_index) if clocks_index is not None else _NoClocks()) as clocks:
        e0.record(stream)
        for _ in range(steps):
            step(timers)
        e1.record(stream)
        barrier()
    ms = max_over_ranks(e0.elapsed_time(e1))
    out = {"cfg": cfg, "wl": wl, "steps": steps, "warmup": warmup, "ms": ms, "nchunks": nchunks,
           "fwd_ms": nchunks * statistics.mean(e[0].elapsed_time(e[1]) for e in timers),   # timed on the last chunk
           "adj_ms": nchunks * statistics.mean(e[2].elapsed_time(e[3]) for e in timers),
           "upd_ms": statistics.mean(e[3].elapsed_time(e[4]) for e in timers),
           # tile / coefficient / finalize kernels of one forward + adjoint over all chunks, + residual,
           # + the epilogue's 2 x (absmax, tv_init, 2 per TV iteration, tv_add, adam)
           "launches": sim.launch_count() * nchunks + nchunks + 2 * (4 + 2 * TV_ITERS),
           "plan": sim.plan, "clocks": clocks.summary(), "e2e": None}
    out["value"] = wl.cell_updates * world * steps / (ms * 1e-3) / 1e9

    # end to end through the host-buffer C-ABI call (H2D of models/wavelet/d_obs, D2H of traces/grads)
    sim.close(); del sim
    if with_e2e:
        del d_obs, res
        torch.cuda.empty_cache()
        p.nshots = wl.nshots
        nb = gprfwi_workspace_bytes_host(p, budget)
        if nb == 0:
            out["e2e"] = {"unavailable": "the whole batch does not fit one gprfwi_gradient_host call"}
        else:
            ws = torch.empty(nb, dtype=torch.uint8, device=dev)
            pin = lambda a: torch.from_numpy(np.ascontiguousarray(a, dtype=np.float32)).pin_memory().numpy()
            h_eps, h_sig, h_w, h_d = pin(wl.eps_r), pin(wl.sigma), pin(wl.wavelet), pin(d_obs_h)
            h_tr = torch.empty((wl.nshots, wl.nt, wl.nrec), dtype=torch.float32).pin_memory().numpy()
            gprfwi_gradient_host(p, h_eps, h_sig, h_w, wl.src_zx, wl.rec_zx, h_d, ws, h_tr)
            barrier()
            # as many end-to-end iterations as timed steps while that stays near a minute, never fewer than 3
            n_e2e = steps if ms <= 60e3 else max(3, min(steps, int(60e3 / (ms / steps))))
            t0 = time.perf_counter()
            for _ in range(n_e2e):
                gprfwi_gradient_host(p, h_eps, h_sig, h_w, wl.src_zx, wl.rec_zx, h_d, ws, h_tr)
            torch.cuda.synchronize()
            dt_e2e = max_over_ranks(time.perf_counter() - t0)
            model_b = wl.nz * wl.nx * 4
            out["e2e"] = {"value": wl.cell_updates * world * n_e2e / dt_e2e / 1e9, "unit": UNIT, "steps": n_e2e,
                          "h2d_bytes_per_step": 2 * model_b + wl.nt * 4 + ntr * 4,
                          "d2h_bytes_per_step": ntr * 4 + 2 * model_b + 8,
                          "call": "gprfwi_gradient_host (pinned host buffers in, host buffers out)"}
            del ws
    torch.cuda.empty_cache()
    return out


def roofline_of(m, peak, peak_src):
    """HBM roofline of the dominant phase (the adjoint sweep with its recompute sweeps) and of the forward
    sweep, from the live CUDA-event times of `m` (run_config's result).  Two fractions, labelled:
      frac_effective_T1  algorithmic bytes of a one-step-per-pass sweep (28 B forward / recompute,
                         32 B adjoint per cell-step) / time / peak.  The kernels fuse T steps per pass, so this
                         can exceed 1: it measures distance from a perfect T = 1 streaming implementation.
      frac_dram          DRAM bytes the kernels really move per cell-step (ncu dram__bytes_read.sum +
                         dram__bytes_write.sum, profiles/dram_traffic.csv) x measured cell-steps/s / peak:
                         the HBM fraction proper, always <= 1."""
    wl, plan = m["wl"], m["plan"]
    cells = wl.nz * wl.nx * wl.nshots
    T = plan["time_block"]
    nlaunch = -(-wl.nt // T)
    recompute = not plan["full_history"]
    # share of the time steps the adjoint phase recomputes: every segment but the last `stored_segments`,
    # whose Ez planes the forward pass kept in spare workspace
    nseg = -(-wl.nt // plan["checkpoint_stride"])
    refrac = (nseg - plan["stored_segments"]) / nseg if recompute else 0.0
    cs = cells * wl.nt                                   # cell-steps of one sweep
    fwd_s, adj_s = m["fwd_ms"] * 1e-3, m["adj_ms"] * 1e-3
    entry, stale = dram_traffic(m["cfg"])
    b = entry or {}
    b_fwd, b_rec, b_adj = b.get("fwd"), b.get("recompute"), b.get("adj")

    fwd_alg = 24.0 + (BYTES_FWD - 24.0) * ((1.0 - refrac) if recompute else 1.0)     # + the Ez planes it keeps
    adj_alg = BYTES_ADJ + BYTES_RECOMPUTE * refrac
    adj_dram = None if b_adj is None or (refrac > 0 and b_rec is None) else b_adj + refrac * (b_rec or 0.0)

    def part(alg, dram, secs):
        d = {"ms_per_sweep": secs * 1e3, "gcell_steps_per_s": cs / secs / 1e9,
             "algorithmic_bytes_per_cell_step_T1": alg, "effective_T1_gbs": alg * cs / secs / 1e9,
             "frac_effective_T1": alg * cs / secs / 1e9 / peak,
             "dram_bytes_per_cell_step": dram, "dram_gbs": None, "frac_dram": None}
        if dram is not None:
            d["dram_gbs"] = dram * cs / secs / 1e9
            d["frac_dram"] = d["dram_gbs"] / peak
        return d

    fwd, adj = part(fwd_alg, b_fwd, fwd_s), part(adj_alg, adj_dram, adj_s)
    it_dram = None
    if fwd["dram_gbs"] is not None and adj["dram_gbs"] is not None:
        it_dram = (b_fwd + adj_dram) * cs / (fwd_s + adj_s) / 1e9
    pair_gbs = (fwd_alg + adj_alg) * cs / (fwd_s + adj_s) / 1e9
    return {"bound": "hbm",
            "kernel": "adj_kernel (+ recompute fwd_kernel sweeps)" if recompute else "adj_kernel",
            "achieved": adj["effective_T1_gbs"], "peak": peak, "unit": "GB/s", "frac": adj["frac_effective_T1"],
            "frac_effective_T1": adj["frac_effective_T1"], "frac_dram": adj["frac_dram"],
            "achieved_dram": adj["dram_gbs"],
            "traffic": None if adj_dram is None else adj_dram * cells * T,
            "traffic_source": None if entry is None else entry.get("source"),
            "traffic_stale": stale,
            "peak_source": peak_src, "steps_per_launch": T,
            "launch_is": "one time block of T steps over all shots (issued as up to 3 concurrent lane launches)",
            "algorithmic_bytes_per_launch": adj_alg * cells * T,
            "avg_launch_us": adj_s * 1e6 / nlaunch,
            "recomputed_fraction_of_steps": refrac,
            "limiter": "issue / latency at 12 warps per SM, not DRAM (ncu: profiles/)",
            "note": "achieved / frac are the contract's algorithmic-bytes figures (T = 1 byte counts, may exceed 1 "
                    "because T steps are fused per pass); frac_dram is the measured-DRAM HBM fraction",
            "adjoint_phase": adj, "forward_sweep": fwd,
            "iteration_effective_T1_gbs": pair_gbs, "iteration_effective_T1_frac_of_8TBs_nominal": pair_gbs / 8000.0,
            "iteration_dram_gbs": it_dram, "iteration_frac_dram": None if it_dram is None else it_dram / peak}


def summary_of(m):
    """Short record of a config timed beside the main one (config.also)."""
    wl = m["wl"]
    peak, peak_src = peaks()
    r = roofline_of(m, peak, peak_src)
    return {"workload": wl.name, "grid": [wl.nz, wl.nx], "nt": wl.nt, "shots_per_gpu": wl.nshots,
            "steps": m["steps"], "warmup": m["warmup"], "value": m["value"], "unit": UNIT,
            "ms_per_step": m["ms"] / m["steps"], "fwd_ms": m["fwd_ms"], "adj_ms": m["adj_ms"],
            "epilogue_ms": m["upd_ms"], "plan": m["plan"], "gpu_launches_per_step": m["launches"],
            "frac_effective_T1": r["frac_effective_T1"], "frac_dram": r["frac_dram"],
            "traffic_stale": r["traffic_stale"]}


def spawn_ranks(args) -> int:
    """`--gpus N` without torchrun: re-execute this script under torch.distributed.run, one rank per GPU."""
    import torch
    have = torch.cuda.device_count() if torch.cuda.is_available() else 0
    if have < args.gpus:
        print(f"bench.py: --gpus {args.gpus} needs {args.gpus} CUDA devices, this host has {have} "
              f"(there is no CPU fallback and ranks never share a GPU)", file=sys.stderr)
        return 2
    import socket
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        port = s.getsockname()[1]
    cmd = [sys.executable, "-m", "torch.distributed.run", "--nnodes=1", f"--nproc-per-node={args.gpus}",
           "--master-addr", "127.0.0.1", "--master-port", str(port), os.path.abspath(__file__)] + sys.argv[1:]
    return subprocess.call(cmd)


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=5)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--config", type=int, default=DEFAULT_CONFIG)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--budget-gb", type=float, default=0.0, help="workspace budget (0 = 92%% of free HBM)")
    ap.add_argument("--n", type=int, default=512, help="config 5: grid is n x n")
    ap.add_argument("--batch", type=int, default=1, help="config 5: shots in the batch (per GPU)")
    ap.add_argument("--nt", type=int, default=0, help="tuning only: cut the number of time steps")
    ap.add_argument("--shots", type=int, default=0, help="tuning only: use the first N shots")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-e2e", action="store_true")
    ap.add_argument("--no-also", action="store_true", help="skip the brief runs of the other configs")
    args = ap.parse_args()
    if args.gpus < 1:
        ap.error("--gpus must be >= 1")
    in_torchrun = "WORLD_SIZE" in os.environ
    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    local_rank = int(os.environ.get("LOCAL_RANK", "0"))

    if args.impl == "reference":       # rank 0 alone runs the oracle; the other ranks exit without work
        if rank == 0:
            wl = load_workload(args.config, args.n, args.batch)
            if args.nt > 0 or args.shots > 0:
                wl = wl.subset(list(range(args.shots or wl.nshots)), nt=args.nt or wl.nt)
            run_reference(args, wl)
        return 0
    if args.gpus > 1 and not in_torchrun:
        return spawn_ranks(args)
    if in_torchrun and world != args.gpus:
        raise SystemExit(f"bench.py: --gpus {args.gpus} but WORLD_SIZE={world}")

    import torch
    import torch.distributed as dist
    from paper_2506_20513_b200 import build
    from paper_2506_20513_b200.dist import shard_shots
    build.build()
    if not torch.cuda.is_available():
        raise SystemExit("bench.py needs a CUDA device (there is no CPU fallback)")
    if local_rank >= torch.cuda.device_count():
        raise SystemExit(f"bench.py: rank {rank} has no GPU of its own ({torch.cuda.device_count()} visible)")
    torch.cuda.set_device(local_rank)
    dev = torch.device("cuda", local_rank)
    if world > 1:
        os.environ.setdefault("NCCL_DEBUG", "INFO")      # the rank / transport lines are the evidence of N ranks
        dist.init_process_group("nccl", device_id=dev)
    env = {"dev": dev, "rank": rank, "world": world}

    def rank_workload(cfg):
        """This rank's contiguous block of the world x shots_per_gpu distinct shots."""
        full = load_workload(cfg, args.n, args.batch, world)
        if args.nt > 0 or args.shots > 0:
            full = full.subset(list(range((args.shots or full.nshots // world) * world)), nt=args.nt or full.nt)
        if world == 1:
            return full
        name = full.name
        sub = full.subset(list(shard_shots(full.nshots, rank, world)))
        sub.name = name
        return sub

    wl = rank_workload(args.config)
    m = run_config(args.config, wl, args.steps, args.warmup, env, args.budget_gb, with_e2e=not args.no_e2e,
                   clocks_index=local_rank)
    also = []
    if not args.no_also and not (args.nt or args.shots):
        for c in ALSO.get(args.config, ()):
            w2 = rank_workload(c)
            k = 10 if 2.0 * w2.nz * w2.nx * w2.nt * w2.nshots < 5e10 else 3
            also.append(summary_of(run_config(c, w2, k, 3, env, 0.0, with_e2e=False)))

    peak, peak_src = peaks()
    roofline = roofline_of(m, peak, peak_src)

    cpu = None
    if rank == 0 and world == 1 and not args.no_cpu_baseline:
        import oracle
        oracle.build()
        ns, nt = oracle_sample_shape(wl)
        shots = sorted({(k * wl.nshots) // ns for k in range(ns)})
        secs, w = oracle_sample(wl, shots, nt)
        cpu = {"value": w / secs / 1e9, "unit": UNIT, "cores": oracle.num_threads(), "kind": "oracle",
               "sample": f"oracle.gradient (forward+adjoint, float64) on shots {shots} of {wl.name}, "
                         f"nt {nt} of {wl.nt}, {secs:.1f} s"}

    if rank == 0:
        line = {"metric": METRIC, "value": m["value"], "unit": UNIT, "n_gpus": world, "steps": args.steps,
                "warmup": m["warmup"], "ms_per_step": m["ms"] / args.steps, "higher_is_better": True,
                "scaling": "weak", "vs_baseline": None, "dtype": "f32", "data": "synthetic",
                "config": {"workload": wl.name, "grid": [wl.nz, wl.nx], "nt": wl.nt, "shots_per_gpu": wl.nshots,
                           "receivers": wl.nrec, "plan": m["plan"], "chunks_per_step": m["nchunks"],
                           "fwd_ms": m["fwd_ms"], "adj_ms": m["adj_ms"], "epilogue_ms": m["upd_ms"],
                           "iteration": "forward, residual+misfit, adjoint, TV term + mask + Adam step + clamps",
                           "s_per_fwi_iteration": m["ms"] / args.steps * 1e-3,
                           "sharding": "shots sharded over ranks, one NCCL all-reduce of the two gradient planes "
                                       "per iteration" if world > 1 else "single GPU",
                           "l2": "inputs larger than L2 (Ez history / checkpoints stream through HBM)",
                           "also": also},
                "clocks": m["clocks"], "e2e": m["e2e"], "gpu_launches": int(m["launches"] * args.steps),
                "roofline": roofline, "cpu_baseline": cpu}
        print(json.dumps(line))
    if world > 1:
        dist.destroy_process_group()
    return 0


if __name__ == "__main__":
    sys.exit(main())
