"""Host-side logic of bench.py (no GPU): rank spawning refuses to fake GPUs, the reference arm's bounded
sample, the ncu traffic table and the two labelled roofline fractions."""
import json
import os
import subprocess
import sys
import types

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
sys.path.insert(0, ROOT)
import bench  # noqa: E402
import gpr_inputs as gi  # noqa: E402


def _run(*argv, timeout=600):
    return subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), *argv], capture_output=True, text=True,
                          timeout=timeout, env={**os.environ, "CUDA_VISIBLE_DEVICES": ""})


def test_gpus_n_without_devices_fails_loudly():
    """`--gpus 2` must start 2 ranks on 2 GPUs or fail: it never runs one rank and prints n_gpus 1."""
    r = _run("--gpus", "2", "--steps", "1")
    assert r.returncode != 0
    assert "needs 2 CUDA devices" in r.stderr and r.stdout.strip() == ""


def test_world_size_must_match_gpus():
    env = {**os.environ, "CUDA_VISIBLE_DEVICES": "", "WORLD_SIZE": "4", "RANK": "0", "LOCAL_RANK": "0"}
    r = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--gpus", "2"], capture_output=True,
                       text=True, timeout=300, env=env)
    assert r.returncode != 0 and "WORLD_SIZE=4" in (r.stderr + r.stdout)


def test_reference_arm_prints_contract_line_on_bounded_sample():
    r = _run("--impl", "reference", "--config", "1", "--steps", "2", "--warmup", "1")
    assert r.returncode == 0, r.stderr
    line = json.loads(r.stdout.strip().splitlines()[-1])
    assert line["impl"] == "reference" and line["unit"] == bench.UNIT and line["metric"] == bench.METRIC
    assert line["cpu_baseline"]["kind"] == "oracle" and line["cpu_baseline"]["value"] == line["value"]
    assert line["e2e"]["h2d_bytes_per_step"] == 0 and line["value"] > 0
    assert line["config"]["workload"] == "config1-tiny"


def test_reference_arm_other_ranks_do_no_work():
    env = {**os.environ, "CUDA_VISIBLE_DEVICES": "", "WORLD_SIZE": "2", "RANK": "1", "LOCAL_RANK": "1"}
    r = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--impl", "reference", "--gpus", "2"],
                       capture_output=True, text=True, timeout=300, env=env)
    assert r.returncode == 0 and r.stdout.strip() == ""


def test_oracle_sample_is_bounded_on_every_config():
    """The reference arm and the cpu_baseline leg must stay inside minutes on the big configs: one sample is
    at most ORACLE_SAMPLE_CELL_UPDATES of oracle work (whole shots at full nt while they fit, else a cut nt)."""
    for wl_shape in ((120, 120, 800, 1), (240, 440, 3000, 20), (540, 1040, 4000, 60), (1060, 2060, 6000, 100),
                     (8192, 8192, 1000, 8)):
        nz, nx, nt, S = wl_shape
        wl = types.SimpleNamespace(nz=nz, nx=nx, nt=nt, nshots=S)
        ns, ntc = bench.oracle_sample_shape(wl)
        assert 1 <= ns <= S and 50 <= ntc <= max(nt, 50)
        assert ns == 1 or ntc == nt
        assert 2.0 * nz * nx * ntc * ns <= max(bench.ORACLE_SAMPLE_CELL_UPDATES, 2.0 * nz * nx * 50)


def test_traffic_table_and_two_labelled_fractions():
    """roofline carries the T = 1-effective fraction (may exceed 1) AND the measured-DRAM fraction (<= 1 for
    any plausible time), and flags a traffic entry captured on another build of the kernels."""
    entry, stale = bench.dram_traffic(4)
    assert entry is not None and entry["adj"] > 0 and entry["recompute"] > 0
    assert stale in (True, False)
    wl = types.SimpleNamespace(nz=1060, nx=2060, nt=6000, nshots=100, name="config4-high-frequency")
    m = {"cfg": 4, "wl": wl, "fwd_ms": 2760.0, "adj_ms": 7160.0,
         "plan": {"time_block": 4, "full_history": 0, "checkpoint_stride": 240, "stored_segments": 0}}
    r = bench.roofline_of(m, 6550.4, "test")
    assert r["bound"] == "hbm" and r["frac"] == r["frac_effective_T1"] and r["frac_effective_T1"] > 1.0
    assert 0.0 < r["frac_dram"] <= 1.0 and r["traffic"] > 0 and r["traffic_stale"] == stale
    assert abs(r["adjoint_phase"]["dram_bytes_per_cell_step"] - (entry["adj"] + entry["recompute"])) < 1e-9
    assert r["forward_sweep"]["frac_dram"] is None or r["forward_sweep"]["frac_dram"] <= 1.0
    # a config with no capture: the fraction is null, not a guess
    assert bench.roofline_of({**m, "cfg": 99}, 6550.4, "test")["frac_dram"] is None


def test_world_workload_has_distinct_shots_per_rank():
    """N ranks sweep N x shots_per_gpu DISTINCT shots, not N copies of the same ones."""
    from paper_2506_20513_b200.dist import shard_shots
    one, two = bench.load_workload(2), bench.load_workload(2, world=2)
    assert two.nshots == 2 * one.nshots and two.nz == one.nz and (two.eps_r == one.eps_r).all()
    a = two.src_zx[list(shard_shots(two.nshots, 0, 2))]
    b = two.src_zx[list(shard_shots(two.nshots, 1, 2))]
    assert len(a) == len(b) == one.nshots
    assert len({tuple(x) for x in a} | {tuple(x) for x in b}) == two.nshots
    assert gi.config5(n=512, batch=4).nshots * 2 == bench.load_workload(5, 512, 4, world=2).nshots
