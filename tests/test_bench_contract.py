"""bench.py's line contract on the CPU: the reference arm (the oracle timed on the host cores -- the one leg that needs no GPU) prints ONE
JSON line with the keys the driver reads, and traffic.json's keys have the shape bench.py looks up."""
import json
import os
import subprocess
import sys

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def test_reference_arm_prints_one_json_line():
    out = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--impl", "reference", "--gpus", "1", "--steps", "2", "--warmup", "3",
                          "--workload", "gelu", "--ref-sample", "48"], capture_output=True, text=True, timeout=600, cwd=ROOT)
    assert out.returncode == 0, out.stderr[-2000:]
    lines = [l for l in out.stdout.splitlines() if l.strip()]
    assert len(lines) == 1
    d = json.loads(lines[0])
    assert d["impl"] == "reference" and d["unit"] == "elements/s" and d["higher_is_better"] is True
    assert d["steps"] == 2 and d["warmup"] == 3 and d["n_gpus"] == 1 and d["vs_baseline"] is None
    assert d["value"] > 0 and abs(d["ms_per_step"] * 1e-3 * d["value"] - 48) < 1e-6 * 48 + 1e-3      # value = sample / time per step
    assert d["config"]["workload"].startswith("gelu n=64 f=12 count=393216")
    assert d["cpu_baseline"]["kind"] == "oracle" and d["cpu_baseline"]["cores"] >= 1 and d["cpu_baseline"]["value"] == d["value"]
    assert d["e2e"] == {"value": d["value"], "unit": "elements/s", "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0}


def test_traffic_keys_match_the_lookup():
    """profiles/traffic.json: '<workload>/v<variant>/<elements per launch>/<kernel>' -> bytes, for every BASELINE tensor"""
    from workloads import specs, tensors
    t = json.load(open(os.path.join(ROOT, "profiles", "traffic.json")))
    assert t and all(isinstance(v, int) and v > 0 for v in t.values())
    for k in t:
        name, v, count, kernel = k.split("/")
        assert name in specs.CONFIGS and v[0] == "v" and int(v[1:]) in (0, 1, 5) and kernel in ("k_eval_p3", "k_eval_sp", "k_gen_vec", "k_gen_bit")
        assert int(count) in (tensors.FULL_COUNT[name], 704512)
    for name in specs.CONFIGS:                                  # the evaluation kernel of every tensor, both constructions
        c = 704512 if name == "silu" else tensors.FULL_COUNT[name]
        assert f"{name}/v0/{c}/k_eval_p3" in t
        assert f"{name}/v1/{tensors.FULL_COUNT[name]}/k_eval_sp" in t
