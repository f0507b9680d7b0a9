"""bench.py contract on the CPU: the reference arm (the oracle on the host cores) prints one JSON line with the keys
the driver reads; the byte model of the roofline matches DESIGN.md section 5."""
import json
import os
import subprocess
import sys

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def test_reference_arm_prints_one_json_line():
    out = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--impl", "reference", "--config", "4",
                          "--level", "5", "--steps", "2", "--warmup", "1", "--cpu-sample-iters", "20"],
                         capture_output=True, text=True, timeout=600, cwd=ROOT)
    assert out.returncode == 0, out.stderr[-2000:]
    lines = [l for l in out.stdout.splitlines() if l.strip()]
    assert len(lines) == 1
    d = json.loads(lines[0])
    assert d["impl"] == "reference" and d["metric"] == "cg_rhs_iterations_per_second" and d["higher_is_better"] is True
    assert d["unit"] == "RHS-iterations/s" and d["value"] > 0 and d["steps"] == 2 and d["ms_per_step"] > 0
    assert d["dtype"] == "f64" and d["data"] == "synthetic" and d["vs_baseline"] is None and d["n_gpus"] == 1
    assert "workload" in d["config"] and "model" not in d["config"]
    cb = d["cpu_baseline"]
    assert cb["kind"] == "oracle" and cb["cores"] >= 1 and cb["value"] == d["value"] and "sample" in cb
    assert d["e2e"] == {"value": d["value"], "unit": d["unit"], "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0}


def test_other_ranks_of_the_reference_arm_do_nothing():
    env = dict(os.environ, RANK="1", WORLD_SIZE="2", LOCAL_RANK="1")
    out = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--impl", "reference", "--gpus", "2"],
                         capture_output=True, text=True, timeout=120, cwd=ROOT, env=env)
    assert out.returncode == 0 and out.stdout.strip() == ""


def test_byte_model():
    sys.path.insert(0, ROOT)
    import bench
    V, nnz, K = 7340033, 51300000, 16
    b = bench.algorithmic_bytes(V, nnz, K, 1)
    matrix = (nnz - V) * 12 + V * 16
    assert b["spmm"] == V * K * 8 * 6 + matrix and b["update"] == V * K * 8 * 3 + V * 16
    assert abs(b["iteration"] / (V * K) - 78.5) < 0.3            # bytes per row and right-hand side
    b2 = bench.algorithmic_bytes(V, nnz, K, 2)
    assert b2["spmm"] == V * K * 8 * 9 + 2 * matrix
