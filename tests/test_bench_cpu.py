"""bench.py on the CPU: the reference arm end to end, and a static check that every function bench.py
calls by a bare name exists (the CUDA arm itself needs a GPU; a missing helper there must not wait for
the GPU box to be found)."""
import ast
import builtins
import json
import os
import subprocess
import sys

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def test_reference_arm_prints_the_contract_line():
    out = subprocess.check_output([sys.executable, os.path.join(ROOT, "bench.py"), "--impl", "reference",
                                   "--steps", "1", "--warmup", "0", "--ref-K", "12"], text=True, cwd=ROOT)
    line = json.loads(out.strip().splitlines()[-1])
    assert line["impl"] == "reference" and line["unit"] == "nonces/s" and line["higher_is_better"] is True
    assert line["e2e"] == {"value": line["value"], "unit": "nonces/s", "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0}
    assert line["cpu_baseline"]["kind"] == "oracle" and line["cpu_baseline"]["cores"] == 1
    assert line["config"]["reference_sample_K"] == 12 and "K=12" in line["config"]["workload"]
    assert line["gpu_launches"] == 0 and line["vs_baseline"] is None


def test_bench_has_every_helper_it_calls():
    sys.path.insert(0, ROOT)
    import bench
    tree = ast.parse(open(os.path.join(ROOT, "bench.py")).read())
    local_defs = {n.name for n in ast.walk(tree) if isinstance(n, (ast.FunctionDef, ast.ClassDef))}
    called = {n.func.id for n in ast.walk(tree) if isinstance(n, ast.Call) and isinstance(n.func, ast.Name)}
    missing = sorted(c for c in called if c not in local_defs and not hasattr(builtins, c) and not hasattr(bench, c))
    assert not missing, missing
    peaks = bench.measured_peaks()
    assert peaks["hbm_gbs"] > 1000 and peaks["sm_max_mhz"] > 1000
    assert set(bench.NCU_TRAFFIC) == {("narrow", 12), ("narrow", 13), ("wide", 13)}
    for row in bench.NCU_TRAFFIC.values():
        assert row["s1"] > 0 and row["s2"] > 0 and row["source"].startswith("profiles/")
        assert os.path.exists(os.path.join(ROOT, row["source"].split(" ")[0]))
    cfg = bench.make_config(34)
    assert cfg["passes"] == 2 and cfg["K"] == 34
    assert bench.whole_job_value(31, 2, 100.0) == 2 * (1 << 31) / 0.1
