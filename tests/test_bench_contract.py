"""bench.py's reference arm (the oracle on the host cores) and its JSON contract, on the Tiny workload (CPU only)."""
import json
import os
import subprocess
import sys

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def test_reference_arm_prints_one_json_line_with_the_contract_keys():
    r = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--impl", "reference", "--workload", "tiny",
                        "--steps", "2", "--warmup", "1"], capture_output=True, text=True, check=True, cwd=ROOT)
    lines = [ln for ln in r.stdout.splitlines() if ln.strip()]
    assert len(lines) == 1
    d = json.loads(lines[0])
    assert d["impl"] == "reference" and d["metric"] == "tLISI+detect snapshot Mpix/s" and d["unit"] == "Mpix/s"
    assert d["n_gpus"] == 1 and d["steps"] == 2 and d["warmup"] == 1 and d["higher_is_better"] is True
    assert d["value"] > 0 and d["ms_per_step"] > 0 and d["vs_baseline"] is None and d["dtype"] == "f64"
    assert d["cpu_baseline"]["kind"] == "oracle" and d["cpu_baseline"]["cores"] >= 1 and d["cpu_baseline"]["sample"]
    assert d["cpu_baseline"]["value"] == d["value"] == d["e2e"]["value"]
    assert d["e2e"]["h2d_bytes_per_step"] == 0 and d["e2e"]["d2h_bytes_per_step"] == 0
    assert "tiny" in d["config"]["workload"] and d["gpu_launches"] == 0


def test_reference_arm_other_ranks_exit_quietly():
    env = dict(os.environ, RANK="1", WORLD_SIZE="2", LOCAL_RANK="1")
    r = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--impl", "reference", "--workload", "tiny",
                        "--steps", "1", "--warmup", "1", "--gpus", "2"], capture_output=True, text=True, env=env, cwd=ROOT)
    assert r.returncode == 0 and r.stdout.strip() == ""


def test_default_workload_is_the_largest_single_gpu_config_and_a_failing_child_is_recorded():
    """BASELINE.json's metric names no config: plain `python bench.py` measures configs[3] (50K x 50K) and embeds the
    other configs; a child that cannot run (no GPU here) becomes an "error" record instead of ending the run."""
    import argparse
    sys.path.insert(0, ROOT)
    import bench
    assert bench.DEFAULT_WORKLOAD == "stream50k" and set(bench.OTHER_CONFIGS) == {"meerkat", "ska_aa2", "imgfreq"}
    import synth
    assert (synth.CONFIGS["stream50k"].H, synth.CONFIGS["stream50k"].L, synth.CONFIGS["stream50k"].cfg_index) == (50000, 4, 4)
    import torch
    if not torch.cuda.is_available():
        rec = bench.sub_record(argparse.Namespace(steps=1, warmup=1), "tiny")
        assert set(rec) == {"error", "command"} and "--workload tiny" in rec["command"]
    assert isinstance(bench.cpu_model(), str) and bench.cpu_model()
