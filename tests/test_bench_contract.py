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


def _synthetic_full_result():
    """a result record with the shape and size of a full default run (28 sweep points, 14 ceilings, 28 + 36 next rows,
    W sweep, per-config CPU points, long provenance strings) and awkward floats"""
    pt = lambda L, prec, lay: {"L": L, "prec": prec, "layout": lay, "W": 4, "footprint_MB": 7247.757312, "us_min": 1060.9123456789,
                               "us_median": 1069.7123456789, "issued": "stream", "GBps": 6831.987654321, "GFLOPps": 3131.123456789,
                               "regime": "HBM-bound", "cold_GBps": float("nan"), "frac_of_copy": 1.0181234567, "frac_of_add_2r1w": 0.98,
                               "cold_frac_of_copy": None, "plan": "pipe depth 3"}
    sweep = [pt(L, pr, lay) for L in (8, 12, 16, 24, 32, 48, 64) for pr in ("f64", "f32") for lay in ("scalar", "vector")]
    rows = ["A5 convert xs->xv", "A5 convert ys->yv", "A5 convert ws->wv", "A1 mul scalar", "A2 mul vector W=4",
            "A3 mul3 vector W=4", "A4 mul_add scalar", "A5 convert zv->zb", "A6 copy zs->zc"]
    ops = [{"row": r, "ms": 1.0788128018, "GBps": 6718.2715107, "GFLOPps": 3079.1, "frac_of_measured_peak": 1.02597225,
            "frac_of_copy": 1.00172784} for r in rows]
    src = "profiles/r03_pipe_kernel_full.md: ncu --set full capture at commit 0123abc (" + "provenance " * 30 + ")"
    return {
        "metric": "su3xsu3_stream_GBps", "value": 6842.20974917474, "unit": "GB/s", "n_gpus": 1, "gpu": "NVIDIA B200", "steps": 20,
        "warmup": 5, "warmup_steps_run": 5, "ms_per_step": 8.474171447753907, "higher_is_better": True, "scaling": "weak",
        "vs_baseline": None, "dtype": "f64", "data": "synthetic",
        "config": {"workload": "BASELINE.json configs[4] top point: 64^4 lattice per GPU (16777216 matrices, 2.416 GB per field), "
                               "fp64 complex, scalar + vector(W=4) layouts, rows A1-A6 per step", "L": 64, "step_bytes": 57982058496,
                   "step_flops": 16911433728, "l2_policy": "inputs larger than L2 (every launch streams >= 4.8 GB; L2 = 133 MB)",
                   "parallelism": "single GPU"},
        "GFLOPps": 1995.6445101759655, "gpu_launches": 180,
        "clocks": {"sm_mhz": 1792.0, "sm_max_mhz": 1965.0, "power_w_max": 847.35, "mem_mhz": 3996.0, "mem_max_mhz": 3996.0,
                   "gpu_name": "NVIDIA B200", "samples": 9, "reasons": ["sw_power_cap"]},
        "e2e": {"value": 242.12505645428155, "host_result_vs_oracle_sampled": {"matrices": 4004, "max_rel_err_A1": 5.18e-16, "ok": True},
                "unit": "GB/s", "h2d_bytes_per_step": 9663676416, "d2h_bytes_per_step": 9663676416, "ms_per_step": 239.47,
                "steps": 5, "api": "su3_mul_host (A1), su3_eval_host (A4, x and y resident) + pinned async copies " * 3,
                "host_result_matches_device": True},
        "roofline": {"bound": "hbm", "kernel": "su3_pipe_kernel<double,W=1,OP_MUL> (row A1, z=x*y fp64 scalar)", "achieved": 6718.27,
                     "peak": 6548.2, "unit": "GB/s", "frac": 1.0259722535553857, "peak_source": "measured (MEASURED_PEAKS.json hbm_gbs)",
                     "algorithmic_bytes_per_launch": 7247757312, "avg_launch_ms": 1.0788, "frac_of_same_run_copy": 1.0017,
                     "pin_rate_peak": 7672.32, "frac_of_pin_rate_peak": 0.8757, "pin_rate_peak_source": "x" * 80, "traffic": 7217163000,
                     "traffic_source": src,
                     "traffic_by_kernel": {"A1": {"traffic": 7217163000, "source": src, "algorithmic_bytes": 7247757312},
                                           "A5": {"traffic": 4830000000, "source": src, "algorithmic_bytes": 4831838208}}},
        "cpu_baseline": {"value": 10.15, "unit": "GB/s", "cores": 16, "kind": "oracle", "sample": "one step = rows A1-A6 on the workload's "
                         "own 64^4 fp64 lattice, all cores, best of 2 passes after a first-touch pass", "ms_per_step": 5711.1,
                         "per_config": [{"config": "cfg%d" % i, "op": "mul", "GBps": 30.49, "GFLOPps": 13.9, "bytes_per_matrix": 432,
                                         "ms": 0.058} for i in range(10)],
                         "stream_triad_GBps": 135.54, "one_thread": {"op": "mul", "sample": "z = x*y", "GBps": 2.369, "GFLOPps": 1.08}},
        "ops": ops, "ceilings_GBps": {"su3_copy": 6706.68, "memcpy_d2d": 6599.66, "su3_add_2r1w": 6955.6, "bar_denominator": 6706.68},
        "ceilings_by_size": [dict(pt(L, pr, "scalar"), su3_copy=6700.1, memcpy_d2d=6600.2) for L in (8, 12, 16, 24, 32, 48, 64) for pr in ("f64", "f32")],
        "convert_f32": [pt(48, "f32", "vector") for _ in range(10)], "wsweep": [pt(48, "f32", "vector") for _ in range(6)],
        "next_rows": {"L": 48, "expr": [dict(pt(48, "f64", "scalar"), program="01*2*3*") for _ in range(34)],
                      "shift": [pt(48, "f64", "vector") for _ in range(32)]},
        "halo": None, "sweep": sweep, "checks": {"vector_result_equals_scalar_result_bitwise": True, "copy_bitwise": True},
        "wall_s_timed_region": 0.1695, "paper_context": {"hardware": "NVIDIA GTX 1080, 288 GB/s peak", "note": "context only " * 20},
    }


def test_headline_record_is_compact_strict_json_with_the_contract_keys(capsys, tmp_path, monkeypatch):
    """the LAST stdout line is what the driver parses: under 4 KB, strict JSON, the keys of the contract; everything
    else goes to stderr as one DETAIL line (round 2's single 36 KB line was not parsed)"""
    sys.path.insert(0, ROOT)
    import bench
    full = _synthetic_full_result()
    assert len(json.dumps(full)) > 30000                                   # the size that broke round 2
    bench.emit(full)
    cap = capsys.readouterr()
    out = [l for l in cap.out.splitlines() if l.strip()]
    assert len(out) == 1 and len(out[0]) < bench.HEADLINE_MAX_BYTES
    bad = lambda c: (_ for _ in ()).throw(ValueError("non-strict constant " + c))
    h = json.loads(out[0], parse_constant=bad)
    for k in ("metric", "value", "unit", "n_gpus", "gpu", "steps", "warmup", "ms_per_step", "higher_is_better", "scaling",
              "vs_baseline", "dtype", "data", "gpu_launches", "config", "clocks", "checks", "roofline", "cpu_baseline", "e2e", "bar"):
        assert k in h, k
    assert h["value"] > 0 and h["metric"] == "su3xsu3_stream_GBps" and h["vs_baseline"] is None
    assert set(h["config"]) >= {"workload", "L", "step_bytes", "step_flops", "l2_policy", "parallelism"}
    rf = h["roofline"]
    assert rf["bound"] == "hbm" and rf["unit"] == "GB/s" and abs(rf["frac"] - rf["achieved"] / rf["peak"]) < 1e-4
    assert rf["traffic"] == 7217163000 and [k["row"] for k in rf["kernels"]] == ["A1", "A5"]
    for k in rf["kernels"]:
        assert set(k) >= {"achieved", "peak", "frac", "algorithmic_bytes_per_launch", "avg_launch_ms", "traffic", "traffic_source"}
    assert rf["kernels"][1]["traffic"] == 4830000000 and rf["kernels"][1]["algorithmic_bytes_per_launch"] == 4831838208
    assert set(h["cpu_baseline"]) >= {"value", "unit", "cores", "kind", "sample", "ms_per_step", "one_thread_GBps", "stream_triad_GBps"}
    assert "per_config" not in h["cpu_baseline"]
    e = h["e2e"]
    assert e["value"] > 0 and e["h2d_bytes_per_step"] == 9663676416 and e["d2h_bytes_per_step"] == 9663676416
    assert e["host_result_matches_device"] is True and e["host_result_vs_oracle_sampled_ok"] is True
    assert len(h["bar"]["points"]) == 8 and all(len(v) == 2 for v in h["bar"]["points"].values())
    for k in ("sweep", "ceilings_by_size", "wsweep", "convert_f32", "next_rows", "ops", "paper_context"):
        assert k not in h
    err = [l for l in cap.err.splitlines() if l.startswith("DETAIL ")]
    assert len(err) == 1
    d = json.loads(err[0][len("DETAIL "):], parse_constant=bad)               # NaN became null
    assert len(d["sweep"]) == 28 and d["sweep"][0]["cold_GBps"] is None and "next_rows" in d and "paper_context" in d
