"""CPU-side checks of bench.py: the N > 1 reduction (gloo, world_size 2), the reference arm and the
level-A byte count."""
import json
import os
import subprocess
import sys

import numpy as np

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _last_json(out):
    lines = [l for l in out.splitlines() if l.startswith("{")]
    assert lines, out
    return json.loads(lines[-1])


def test_two_rank_reduction_is_max_time_sum_units():
    """world_size 2 over gloo: whole-job time = MAX over ranks, units = SUM (bench.py contract)."""
    cmd = [sys.executable, "-m", "torch.distributed.run", "--nnodes=1", "--nproc-per-node", "2",
           "--master-addr", "127.0.0.1", "--master-port", "29731", os.path.join(ROOT, "bench.py"),
           "--gpus", "2", "--selftest-dist"]
    r = subprocess.run(cmd, capture_output=True, text=True, timeout=300, cwd=ROOT)
    assert r.returncode == 0, r.stderr[-2000:]
    j = _last_json(r.stdout)
    assert j["n_gpus"] == 2 and j["ms"] == 20.0 and j["units"] == 3000.0
    assert abs(j["value"] - 3000.0 / 0.020) < 1e-6


def test_reference_arm_prints_contract_line():
    r = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--impl", "reference", "--steps", "1",
                        "--warmup", "0", "--ref-cells", "40"], capture_output=True, text=True, timeout=600, cwd=ROOT)
    assert r.returncode == 0, r.stderr[-2000:]
    j = _last_json(r.stdout)
    assert j["impl"] == "reference" and j["value"] > 0 and j["unit"] == "CV-steps/s"
    assert j["cpu_baseline"]["kind"] == "oracle" and j["cpu_baseline"]["cores"] >= 1
    assert j["e2e"]["h2d_bytes_per_step"] == 0 and j["gpu_launches"] == 0


def test_level_a_bytes_match_the_survey_figure():
    """C3 cell = 505*48 + 63*4 + 80 + 50*20 = 25,572 B per cell-step (the soma has one
    child, so it is the first CV of the root branch)."""
    sys.path.insert(0, ROOT)
    import bench
    from paper_1901_07454_b200 import workloads as W
    m = W.config3(n_cells=10)
    assert bench.algorithmic_bytes_per_grid_step(m) == 10 * 25572
