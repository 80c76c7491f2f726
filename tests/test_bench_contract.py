"""The parts of bench.py's contract that can be checked without a GPU: the reference arm (the oracle timed on
the host cores) prints exactly one JSON line with the agreed keys, idle ranks print nothing, and our own arm
refuses to run without a CUDA device instead of falling back to anything."""
import json
import os
import subprocess
import sys

import torch

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def run(args, env=None):
    e = dict(os.environ)
    e.update(env or {})
    return subprocess.run([sys.executable, os.path.join(ROOT, "bench.py")] + args, capture_output=True, text=True, env=e,
                          timeout=600)


def test_reference_arm_prints_one_json_line_with_the_contract_keys():
    r = run(["--impl", "reference", "--steps", "2", "--warmup", "1", "--L", "8"])
    assert r.returncode == 0, r.stderr
    lines = [l for l in r.stdout.splitlines() if l.strip()]
    assert len(lines) == 1
    d = json.loads(lines[0])
    assert d["impl"] == "reference" and d["metric"] == "su3xsu3_stream_GBps" and d["unit"] == "GB/s"
    assert d["steps"] == 2 and d["warmup"] == 1 and d["higher_is_better"] is True and d["vs_baseline"] is None
    assert d["value"] > 0 and d["ms_per_step"] > 0 and d["dtype"] == "f64" and d["data"] == "synthetic"
    assert d["cpu_baseline"]["kind"] == "oracle" and d["cpu_baseline"]["cores"] >= 1 and d["cpu_baseline"]["value"] == d["value"]
    assert d["e2e"] == {"value": d["value"], "unit": "GB/s", "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0}
    assert "workload" in d["config"] and d["config"]["same_config"] is True and d["config"]["sample_L"] == 8


def test_reference_arm_other_ranks_exit_quietly():
    r = run(["--impl", "reference", "--gpus", "2", "--steps", "1", "--warmup", "0", "--L", "8"],
            env={"RANK": "1", "WORLD_SIZE": "2", "LOCAL_RANK": "1"})
    assert r.returncode == 0 and r.stdout.strip() == ""


def test_own_arm_has_no_cpu_fallback():
    if torch.cuda.is_available():
        return
    r = run(["--steps", "1", "--L", "8"])
    assert r.returncode != 0 and "no CPU fallback" in r.stderr and r.stdout.strip() == ""


def test_oracle_step_and_cpu_baseline_leg_on_a_small_lattice():
    """the cpu_baseline leg (the oracle timed with first-touched outputs, per-config points, 1 thread, STREAM triad)"""
    import types
    sys.path.insert(0, ROOT)
    import bench
    import su3gen
    L = 8
    n = L ** 4
    host = {}
    for name, fid in (("x", 0), ("y", 1), ("w", 2), ("v", 3)):
        a = (su3gen.gaussian_field if name == "v" else su3gen.su3_field)(su3gen.config_seed(5), fid, n)
        host[name] = torch.from_numpy(a.reshape(-1))
    cpu = bench.run_cpu_baseline(types.SimpleNamespace(L=L), host)
    assert cpu["kind"] == "oracle" and cpu["value"] > 0 and cpu["cores"] >= 1 and "8^4" in cpu["sample"]
    names = [p["config"] for p in cpu["per_config"]]
    assert any(nm.startswith("cfg1") for nm in names) and all(p["GBps"] > 0 for p in cpu["per_config"])
    assert cpu["one_thread"]["GBps"] > 0 and cpu["stream_triad_GBps"] > 0
    import oracle
    assert oracle.num_threads() == cpu["cores"]          # the 1-thread leg restored the thread count
    assert bench.ncu_traffic(7)[0] is None
