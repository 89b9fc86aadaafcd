"""bench.py --impl reference on CPU: the oracle timed on the host cores, one JSON line with the contract's keys
(the arm needs no GPU; configs[0] keeps it to seconds)."""
import json
import os
import subprocess
import sys

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def test_reference_arm_prints_the_contract_line():
    out = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--impl", "reference", "--config", "0", "--steps", "3",
                          "--warmup", "3"], capture_output=True, text=True, timeout=600, cwd=ROOT)
    assert out.returncode == 0, out.stderr[-2000:]
    line = json.loads(out.stdout.strip().splitlines()[-1])
    assert line["impl"] == "reference" and line["metric"] == "superiorization iterations/sec" and line["unit"] == "iterations/s"
    assert line["value"] > 0 and line["steps"] == 3 and line["warmup"] == 3 and line["higher_is_better"] is True
    assert line["cpu_baseline"]["kind"] == "oracle" and line["cpu_baseline"]["cores"] >= 1
    assert "iterations 3..5 from x0" in line["cpu_baseline"]["sample"]        # the window our arm times: W warm-up, then K
    assert line["e2e"] == {"value": line["value"], "unit": "iterations/s", "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0}
    assert line["config"]["workload"].startswith("configs[0]") and line["vs_baseline"] is None
    # `config` states the workload from the plan and the flags alone (bench.workload_config): the object our arm prints too
    for k in ("n_voxels", "n_spots", "nnz_per_matrix", "n_labelled_voxels", "lambda", "beta0", "a", "form", "ams_form", "l2", "parallelism"):
        assert k in line["config"]
    assert line["config"]["form"] == "superiorized" and line["config"]["l2"].startswith("L2-resident")


@pytest.mark.gpu
def test_both_arms_state_the_same_config():
    """The driver divides our arm's value by the reference arm's: both lines must name the same workload, key for key."""
    lines = []
    for impl in ("reference", "ours"):
        out = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--impl", impl, "--config", "0", "--steps", "3", "--warmup", "3",
                              "--no-cpu-baseline", "--no-forms"], capture_output=True, text=True, timeout=900, cwd=ROOT)
        assert out.returncode == 0, out.stderr[-2000:]
        lines.append(json.loads(out.stdout.strip().splitlines()[-1]))
    ref, ours = lines
    assert ref["config"] == ours["config"]
    assert (ref["metric"], ref["unit"], ref["higher_is_better"], ref["steps"], ref["warmup"]) == \
           (ours["metric"], ours["unit"], ours["higher_is_better"], ours["steps"], ours["warmup"])
    assert ours["plan"]["block_rows"] in (1, 2, 4) and ours["gpu_launches"] > 0 and ref["gpu_launches"] == 0


def test_reference_arm_other_ranks_exit_quietly():
    env = dict(os.environ, RANK="1", WORLD_SIZE="2", LOCAL_RANK="1")
    out = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--impl", "reference", "--config", "0", "--gpus", "2"],
                         capture_output=True, text=True, timeout=600, cwd=ROOT, env=env)
    assert out.returncode == 0 and out.stdout.strip() == ""
