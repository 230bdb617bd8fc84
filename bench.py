#!/usr/bin/env python
"""bench.py -- forward+adjoint FDTD throughput of libgprfwi on BASELINE.json's configs.

A "step" is one pass of the whole hot path over one batch of synthetic input: coefficient build,
nt forward steps (H+E+CPML+source+receivers+history), residual, nt adjoint steps with gradient
accumulation, chain rule.  Default workload: BASELINE.json configs[1] (paper-scale synthetic,
240x440 full grid, nt=3000, 20 shots, 100 receivers, full Ez history in HBM).

    python bench.py [--gpus N] [--steps K] [--warmup W] [--config 2|3|4|1] [--impl ours|reference]

Prints ONE JSON line (rank 0).  `--impl reference` times the float64 CPU oracle (oracle/) instead.
"""
from __future__ import annotations

import argparse
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


def load_workload(cfg: int, n: int = 512, batch: int = 1):
    if cfg == 5:
        return gi.config5(n=n, batch=batch)
    return {1: gi.config1, 2: gi.config2, 3: gi.config3, 4: gi.config4}[cfg]()


def peaks():
    path = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(path):
        with open(path) as f:
            return float(json.load(f)["hbm_gbs"]), "measured (MEASURED_PEAKS.json, burst copy)"
    return 6650.0, "fallback (B200_PROFILING.md)"


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


def oracle_sample(wl, shots):
    """Oracle forward+adjoint on a few shots of the workload; returns (seconds, cell_updates)."""
    import oracle
    from helpers import problem
    sub = wl.subset(shots)
    res = gi.random_residual(sub, 1.0)
    t0 = time.perf_counter()
    oracle.gradient(problem(sub), sub.eps_r, sub.sigma, res)
    return time.perf_counter() - t0, sub.cell_updates


def run_reference(args, wl):
    import oracle
    oracle.build()
    per_step_shots = [0]
    for _ in range(args.warmup):
        oracle_sample(wl.subset([0], nt=min(wl.nt, 200)), [0])
    times, work = [], 0
    for k in range(args.steps):
        t, w = oracle_sample(wl, [(k * 7) % wl.nshots])
        times.append(t); work += w
    total = sum(times)
    val = work / total / 1e9
    sample = f"{args.steps} steps x 1 shot of {wl.name} (full grid, full nt), float64, OpenMP over rows"
    line = {"impl": "reference", "metric": METRIC, "value": val, "unit": UNIT, "n_gpus": args.gpus,
            "steps": args.steps, "warmup": args.warmup, "ms_per_step": 1e3 * total / args.steps,
            "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f64",
            "data": "synthetic", "config": {"workload": wl.name, "sample": sample},
            "cpu_baseline": {"value": val, "unit": UNIT, "cores": oracle.num_threads(), "kind": "oracle",
                             "sample": sample},
            "e2e": {"value": val, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
            "gpu_launches": 0}
    print(json.dumps(line))


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=20)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--config", type=int, default=2)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--budget-gb", type=float, default=0.0, help="workspace budget (0 = 92%% of free HBM)")
    ap.add_argument("--n", type=int, default=512, help="config 5: grid is n x n")
    ap.add_argument("--batch", type=int, default=1, help="config 5: shots in the batch")
    ap.add_argument("--nt", type=int, default=0, help="tuning only: cut the number of time steps")
    ap.add_argument("--shots", type=int, default=0, help="tuning only: use the first N shots")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-e2e", action="store_true")
    args = ap.parse_args()
    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    local_rank = int(os.environ.get("LOCAL_RANK", "0"))

    wl = load_workload(args.config, args.n, args.batch)
    if args.nt > 0 or args.shots > 0:
        wl = wl.subset(list(range(args.shots or wl.nshots)), nt=args.nt or wl.nt)
    if args.impl == "reference":
        if rank == 0:
            run_reference(args, wl)
        return 0

    import torch
    import torch.distributed as dist
    from paper_2506_20513_b200 import (Simulation, build, split_batch, gprfwi_gradient_host, gprfwi_residual, gprfwi_update,
                                       gprfwi_update_workspace_bytes, gprfwi_workspace_bytes,
                                       gprfwi_workspace_bytes_host, make_params, make_update_params)
    from paper_2506_20513_b200.dist import allreduce_gradients
    build.build()
    if not torch.cuda.is_available():
        raise SystemExit("bench.py needs a CUDA device (there is no CPU fallback)")
    torch.cuda.set_device(local_rank)
    dev = torch.device("cuda", local_rank)
    if world > 1:
        dist.init_process_group("nccl", device_id=dev)

    p = make_params(nz=wl.nz, nx=wl.nx, dx=wl.dx, dt=wl.dt, nt=wl.nt, npml=wl.npml, pml_order=wl.pml_order,
                    pml_sigma_max=wl.pml_sigma_max, pml_kappa_max=wl.pml_kappa_max,
                    pml_alpha_max=wl.pml_alpha_max, nshots=wl.nshots, nrec=wl.nrec)
    free, _total = torch.cuda.mem_get_info(dev)
    ntr = wl.nshots * wl.nt * wl.nrec
    budget = int(args.budget_gb * 1e9) if args.budget_gb > 0 else int(free * 0.92) - 3 * ntr * 4
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
    rng = np.random.Generator(np.random.PCG64(wl.seed + 99))
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
    upd = make_update_params(step=1, lr_eps_r=1e-3, lr_sigma=1e-6, tv_iters=10, mask_rows=wl.npml + 7)

    def step(timers=None):
        ev = [torch.cuda.Event(enable_timing=True) for _ in range(4)] if timers is not None else None
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
            ev.append(torch.cuda.Event(enable_timing=True)); ev[4].record(stream)
            timers.append(ev)

    def barrier():
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    for _ in range(max(args.warmup, 3)):
        step()
    barrier()
    timers = []
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    with ClockSampler(local_rank) as clocks:
        e0.record(stream)
        for _ in range(args.steps):
            step(timers)
        e1.record(stream)
        barrier()
    ms = e0.elapsed_time(e1)
    if world > 1:
        t = torch.tensor([ms], device=dev)
        dist.all_reduce(t, op=dist.ReduceOp.MAX)
        ms = float(t.item())
    fwd_ms = nchunks * statistics.mean(e[0].elapsed_time(e[1]) for e in timers)       # timed on the last chunk
    adj_ms = nchunks * statistics.mean(e[2].elapsed_time(e[3]) for e in timers)
    upd_ms = statistics.mean(e[3].elapsed_time(e[4]) for e in timers)
    launches = sim.launch_count() * nchunks   # kernels of one forward + adjoint over all chunks
    plan = sim.plan
    cells = wl.nz * wl.nx * wl.nshots
    work = wl.cell_updates * world
    value = work * args.steps / (ms * 1e-3) / 1e9

    # roofline of the dominant kernel (adjoint: 32 B per cell-step algorithmic, T = 1 figure of
    # SURVEY.md 8(d)) from live CUDA-event times.  One launch fuses T = plan["time_block"] steps, so
    # the launch count per sweep is ceil(nt / T) and the algorithmic bytes per launch are T * 32 B * cells.
    peak, peak_src = peaks()
    T = plan["time_block"]
    nlaunch = -(-wl.nt // T)
    recompute = not plan["full_history"]
    # share of the time steps the adjoint phase recomputes: every segment but the last `stored_segments`,
    # whose Ez planes the forward pass kept in spare workspace
    nseg = -(-wl.nt // plan["checkpoint_stride"])
    refrac = (nseg - plan["stored_segments"]) / nseg if recompute else 0.0
    adj_bytes = cells * BYTES_ADJ * wl.nt / nlaunch
    adj_launch_us = adj_ms * 1e3 / (nlaunch * (1.0 + refrac))              # recompute launches interleave
    achieved = (cells * (BYTES_ADJ + BYTES_RECOMPUTE * refrac) * wl.nt) / (adj_ms * 1e-3) / 1e9
    fwd_bytes = cells * (24.0 + (BYTES_FWD - 24.0) * (1.0 - refrac if recompute else 1.0)) * wl.nt / nlaunch   # + Ez planes kept
    fwd_launch_us = fwd_ms * 1e3 / nlaunch
    # dram__bytes_read.sum + dram__bytes_write.sum of the adjoint kernel per time block, from the
    # `ncu --set full` capture summarised in profiles/r01_v4_README.md (one lane launch of 6 shots moved
    # 24.8 MB; scaled to the 20 shots of a block).  Config 3: adjoint 521.5 MB + recompute sweep 265.7 MB per
    # lane launch of 20 shots, three lanes per block (same README).  Config 4 (profiles/r01_v5_README.md):
    # adjoint 1771 MB + recompute sweep 1411 MB per lane launch of 17 shots, scaled to the 100 shots of a block.
    traffic = {2: 82.7e6, 3: 2361.6e6, 4: 18.72e9}.get(args.config) if not (args.nt or args.shots) else None
    pair_gbs = (fwd_bytes + adj_bytes + cells * BYTES_RECOMPUTE * refrac * wl.nt / nlaunch) \
        * nlaunch / ((fwd_ms + adj_ms) * 1e-3) / 1e9
    roofline = {"bound": "hbm", "kernel": "adj_kernel (+recompute fwd_kernel)" if recompute else "adj_kernel",
                "achieved": achieved, "peak": peak, "unit": "GB/s", "frac": achieved / peak, "traffic": traffic,
                "peak_source": peak_src, "steps_per_launch": T,
                "launch_is": "one time block of T steps over all shots (issued as up to 3 concurrent lane launches)",
                "algorithmic_bytes_per_launch": adj_bytes, "avg_launch_us": adj_launch_us,
                "recomputed_fraction_of_steps": refrac,
                "note": "algorithmic bytes are the one-step-per-pass figures (32 B adj, 28 B fwd per cell-step); "
                        "the kernels fuse T steps per pass, so frac can exceed what a T=1 sweep could reach",
                "forward": {"kernel": "fwd_kernel", "achieved": fwd_bytes / (fwd_launch_us * 1e-6) / 1e9,
                            "avg_launch_us": fwd_launch_us,
                            "frac": fwd_bytes / (fwd_launch_us * 1e-6) / 1e9 / peak},
                "pair_effective_gbs": pair_gbs, "frac_of_8TBs_nominal": pair_gbs / 8000.0}

    # end to end through the host-buffer C-ABI call (H2D of models/wavelet/d_obs, D2H of traces/grads)
    e2e = None
    if not args.no_e2e:
        sim.close(); del sim
        torch.cuda.empty_cache()
        nb = gprfwi_workspace_bytes_host(p, budget)
        ws = torch.empty(nb, dtype=torch.uint8, device=dev)
        pin = lambda a: torch.from_numpy(np.ascontiguousarray(a, dtype=np.float32)).pin_memory().numpy()
        h_eps, h_sig, h_w, h_d = pin(wl.eps_r), pin(wl.sigma), pin(wl.wavelet), pin(d_obs_h)
        h_tr = torch.empty((wl.nshots, wl.nt, wl.nrec), dtype=torch.float32).pin_memory().numpy()
        gprfwi_gradient_host(p, h_eps, h_sig, h_w, wl.src_zx, wl.rec_zx, h_d, ws, h_tr)
        barrier()
        t0 = time.perf_counter()
        for _ in range(args.steps):
            gprfwi_gradient_host(p, h_eps, h_sig, h_w, wl.src_zx, wl.rec_zx, h_d, ws, h_tr)
        torch.cuda.synchronize()
        dt_e2e = time.perf_counter() - t0
        if world > 1:
            t = torch.tensor([dt_e2e], device=dev)
            dist.all_reduce(t, op=dist.ReduceOp.MAX)
            dt_e2e = float(t.item())
        model_b = wl.nz * wl.nx * 4
        e2e = {"value": work * args.steps / dt_e2e / 1e9, "unit": UNIT,
               "h2d_bytes_per_step": 2 * model_b + wl.nt * 4 + ntr * 4,
               "d2h_bytes_per_step": ntr * 4 + 2 * model_b + 8}

    cpu = None
    if rank == 0 and world == 1 and not args.no_cpu_baseline:
        import oracle
        oracle.build()
        shots = sorted({(k * wl.nshots) // 8 for k in range(8)}) if args.config <= 2 else [0]
        sub = wl if args.config <= 2 else wl.subset(list(range(wl.nshots)), nt=min(wl.nt, 400))
        secs, w = oracle_sample(sub, shots)
        cpu = {"value": w / secs / 1e9, "unit": UNIT, "cores": oracle.num_threads(), "kind": "oracle",
               "sample": f"oracle.gradient (forward+adjoint, float64) on shots {shots} of {sub.name}, "
                         f"{secs:.1f} s"}

    if rank == 0:
        line = {"metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps,
                "warmup": max(args.warmup, 3), "ms_per_step": ms / args.steps, "higher_is_better": True,
                "scaling": "weak", "vs_baseline": None, "dtype": "f32", "data": "synthetic",
                "config": {"workload": wl.name, "grid": [wl.nz, wl.nx], "nt": wl.nt, "shots_per_gpu": wl.nshots,
                           "receivers": wl.nrec, "plan": plan, "chunks_per_step": nchunks, "fwd_ms": fwd_ms, "adj_ms": adj_ms, "epilogue_ms": upd_ms,
                           "iteration": "forward, residual+misfit, adjoint, TV term + mask + Adam step + clamps",
                           "s_per_fwi_iteration": ms / args.steps * 1e-3,
                           "l2": "inputs larger than L2 (Ez history / checkpoints stream through HBM)"},
                "clocks": clocks.summary(), "e2e": e2e, "gpu_launches": int((launches + 1) * args.steps),
                "roofline": roofline, "cpu_baseline": cpu}
        print(json.dumps(line))
    if world > 1:
        dist.destroy_process_group()
    return 0


if __name__ == "__main__":
    sys.exit(main())
