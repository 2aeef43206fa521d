"""bench.py contract on CPU: the reference arm (the oracle on host cores) prints one JSON line with the keys the
driver reads; no GPU needed."""
import json
import os
import subprocess
import sys

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def test_reference_arm_prints_contract_line():
    import time
    t0 = time.perf_counter()
    out = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--impl", "reference", "--steps", "2",
                          "--warmup", "1"], capture_output=True, text=True, timeout=900, cwd=ROOT)
    wall = time.perf_counter() - t0
    assert out.returncode == 0, out.stderr[-2000:]
    line = json.loads(out.stdout.strip().splitlines()[-1])
    # the line reports the steps and warm-ups it really ran: they must fit into the run's wall clock
    assert line["steps"] == 2 and line["warmup"] == 1
    assert (line["steps"] + line["warmup"]) * line["ms_per_step"] * 1e-3 <= wall
    assert set(line["call_ms"]) == {"cbct_fp", "cbct_bp_adjoint", "cbct_bp_fdk"}
    assert line["backprojection"]["adjoint_gvoxel_views_per_s"] > 0 and line["backprojection"]["fdk_gvoxel_views_per_s"] > 0
    assert line["impl"] == "reference" and line["higher_is_better"] is True
    for key in ("metric", "value", "unit", "n_gpus", "steps", "warmup", "ms_per_step", "scaling", "vs_baseline",
                "dtype", "data", "config", "cpu_baseline", "e2e"):
        assert key in line, key
    assert line["value"] > 0 and line["dtype"] == "f64" and line["vs_baseline"] is None
    assert line["cpu_baseline"]["kind"] == "oracle" and line["cpu_baseline"]["cores"] >= 1
    assert line["e2e"]["h2d_bytes_per_step"] == 0 and line["e2e"]["d2h_bytes_per_step"] == 0
    assert line["config"]["workload"] == "multichannel_256"


def test_reference_arm_other_ranks_exit_quietly():
    env = dict(os.environ, RANK="1", WORLD_SIZE="2", LOCAL_RANK="1")
    out = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--impl", "reference", "--gpus", "2"],
                         capture_output=True, text=True, timeout=120, cwd=ROOT, env=env)
    assert out.returncode == 0 and out.stdout.strip() == ""


def test_work_models_are_what_design_states():
    """bench.py's algorithmic work per step (DESIGN.md s.7): 32 B per forward sample, 16 B per FDK voxel-view, and for
    the gather adjoint 8 terms per sample, each one accumulate plus its share of an 8-instruction weight."""
    sys.path.insert(0, ROOT)
    import bench
    m = bench.work_models(C=8, n_samples=1000, n_vv=500, rotations=4, mirror=True)
    assert m["fp"]["work"] == 32.0 * 8 * 1000 and m["fdk"]["work"] == 16.0 * 8 * 500
    assert m["adjoint"]["sharing"] == 64 and m["adjoint"]["work"] == 8.0 * 8 * 1000 * (1 + 8 / 64)
    m1 = bench.work_models(C=1, n_samples=1000, n_vv=500, rotations=1, mirror=False)
    assert m1["adjoint"]["work"] == 8.0 * 1000 * 9.0 and m1["adjoint"]["bound"] == "alu"
