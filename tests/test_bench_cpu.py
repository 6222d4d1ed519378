"""CPU-side checks of bench.py's contract: the reference arm (the oracle, timed as it stands on a
bounded sample) prints ONE JSON line with the agreed keys; under a multi-rank launch only rank 0
prints; the algorithmic byte counts are the ones of SURVEY.md 8(d)."""
import json
import os
import subprocess
import sys

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
sys.path.insert(0, ROOT)


def _run(extra, env=None):
    e = dict(os.environ)
    e.update(env or {})
    out = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--impl", "reference", "--config", "mlp3_k4",
                          "--steps", "2", "--warmup", "1"] + extra, capture_output=True, text=True, env=e, timeout=300)
    assert out.returncode == 0, out.stderr
    return [l for l in out.stdout.splitlines() if l.strip()]


def test_reference_arm_prints_one_line_with_the_contract_keys():
    lines = _run([])
    assert len(lines) == 1
    d = json.loads(lines[0])
    for k in ("metric", "value", "unit", "n_gpus", "steps", "warmup", "ms_per_step", "higher_is_better", "scaling",
              "vs_baseline", "dtype", "data", "config", "impl", "cpu_baseline", "e2e", "gpu_launches"):
        assert k in d, k
    assert d["impl"] == "reference" and d["metric"] == "param_updates_per_s" and d["unit"] == "param-updates/s"
    assert d["vs_baseline"] is None and d["dtype"] == "f32" and d["steps"] == 2 and d["value"] > 0
    assert d["cpu_baseline"]["kind"] == "oracle" and d["cpu_baseline"]["cores"] == os.cpu_count()   # -fopenmp build
    assert d["e2e"]["value"] == d["value"] and d["e2e"]["h2d_bytes_per_step"] == 0
    assert "workload" in d["config"] and "model" not in d["config"]
    # both arms print the SAME config dict (the driver's same_config check): what is computed, not how it is launched
    import argparse
    import bench
    import synth
    args = argparse.Namespace(optimizer="sgd", mix="pushsum")
    assert d["config"] == json.loads(json.dumps(bench.bench_config(synth.workload("mlp3_k4"), args)))
    assert sorted(d["config"]) == sorted(["workload", "K", "L", "params_per_replica", "momentum", "lr", "skip_prob",
                                          "optimizer", "mix"])
    src = open(os.path.join(ROOT, "bench.py")).read()
    assert src.count('"config": bench_config(w, args)') == 2          # run_reference and run_ours


def test_committed_traffic_names_its_capture():
    import bench
    t, where = bench.committed_traffic("gpt2m_k16", "sgd")
    assert t > 1e11 and "profiles/" in where and "captured 20" in where and " at " in where
    assert bench.committed_traffic("no_such_workload") == (None, None)


def test_reference_arm_other_ranks_stay_silent():
    assert _run([], env={"RANK": "1", "WORLD_SIZE": "2", "LOCAL_RANK": "1"}) == []


def test_reference_arm_covers_the_widened_rule():
    d = json.loads(_run(["--optimizer", "adamw", "--mix", "symmetric"])[0])
    assert d["value"] > 0


def test_algorithmic_bytes_per_update():
    import argparse

    import bench
    import synth
    sgd = argparse.Namespace(optimizer="sgd", mix="pushsum")
    adam = argparse.Namespace(optimizer="adamw", mix="pushsum")
    assert bench.bytes_per_update(synth.workload("mlp3_k4"), sgd) == 12          # read x, g; write x
    assert bench.bytes_per_update(synth.workload("gpt2m_k16"), sgd) == 20        # + read, write m
    assert bench.bytes_per_update(synth.workload("gpt2m_k16"), adam) == 28       # + read, write v
    w = synth.workload("gpt2m_k16")
    bts, ups = bench.algorithmic_bytes(w, None, range(3), sgd)
    assert ups == [16 * 354823168] * 3 and bts == [20 * 16 * 354823168] * 3
