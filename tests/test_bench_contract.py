"""bench.py prints ONE JSON line with the keys the driver and the judge read (both arms)."""
import json
import os
import subprocess
import sys

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
BASE_KEYS = {"metric", "value", "unit", "n_gpus", "steps", "warmup", "ms_per_step", "higher_is_better", "scaling",
             "vs_baseline", "dtype", "data", "config", "e2e", "cpu_baseline"}


def _run(args, timeout=600):
    res = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py")] + args, capture_output=True, text=True,
                         timeout=timeout, cwd=ROOT)
    assert res.returncode == 0, res.stderr[-2000:]
    lines = [l for l in res.stdout.splitlines() if l.strip()]
    assert len(lines) == 1, f"bench.py must print exactly one line, got {len(lines)}"
    return json.loads(lines[0])


@pytest.mark.parametrize("tuning", ["with-ut", "no-ut"])
def test_reference_arm_line(tuning):
    """--impl reference times the oracle on the host cores: no GPU needed."""
    d = _run(["--impl", "reference", "--steps", "1", "--warmup", "0", "--events", "60", "--tuning", tuning])
    assert BASE_KEYS <= set(d) and d["impl"] == "reference"
    assert d["metric"] == "events_per_s" and d["unit"] == "events/s" and d["higher_is_better"] is True
    assert d["value"] > 0 and d["vs_baseline"] is None and d["data"] == "synthetic" and d["dtype"] == "f32"
    assert d["cpu_baseline"]["kind"] == "oracle" and d["cpu_baseline"]["cores"] >= 1 and d["cpu_baseline"]["value"] == d["value"]
    assert d["e2e"] == {"value": d["value"], "unit": "events/s", "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0}
    assert "workload" in d["config"] and "model" not in d["config"]


@pytest.mark.gpu
@pytest.mark.parametrize("tuning", ["with-ut", "no-ut"])
def test_gpu_arm_line(tuning):
    d = _run(["--steps", "3", "--warmup", "3", "--events", "400", "--cpu-events", "100", "--tuning", tuning])
    assert BASE_KEYS | {"roofline", "clocks", "gpu_launches"} <= set(d)
    assert d["metric"] == "events_per_s" and d["n_gpus"] == 1 and d["steps"] == 3 and d["warmup"] >= 3
    assert d["value"] > 0 and d["ms_per_step"] > 0 and d["scaling"] == "weak" and d["vs_baseline"] is None
    assert d["gpu_launches"] == 4 * 3
    e = d["e2e"]
    assert e["value"] > 0 and e["value"] < d["value"] and e["h2d_bytes_per_step"] > 0 and e["d2h_bytes_per_step"] > 0
    r = d["roofline"]
    # top level = the HBM roofline BASELINE.json's metric names.  ncu's DRAM bytes and instruction counts describe the
    # full configs[3] batch on the stamped source only (profiles/dominant_kernel_traffic*.txt): on this small batch
    # "traffic" and "issue_utilisation" must be null, never a stale number
    assert r["bound"] == "hbm" and r["unit"] == "GB/s" and 0 < r["frac"] < 1 and r["achieved"] > 0 and r["peak"] > 0
    assert r["traffic"] is None and r["algorithmic_bytes_per_launch"] > 0 and d["issue_utilisation"] is None
    # the algorithmic ALU fraction comes from the committed model evaluated on this batch's own work counters
    assert 0 < d["alu_algorithmic_frac"] < 1
    c = d["alu_model"]["counters"]
    assert c["tracks"] == d["config"]["tracks_per_step_per_gpu"] and c["window_hits"] > c["doublets_passing"] > 0
    assert c["doublets_evaluated"] >= c["doublets_passing"] and c["triplets_passing"] >= c["triplets_kept"] >= c["accepted_candidates"] > 0
    assert abs(sum(v for k, v in d["alu_model"]["lane_ops_per_step"].items() if k != "total") - d["alu_model"]["lane_ops_per_step"]["total"]) < 1
    c = d["cpu_baseline"]
    assert c["kind"] == "oracle" and c["cores"] == 1 and c["value"] > 0 and "sample" in c
    assert d["oracle_check"]["equal"] is True
    assert set(d["clocks"]) >= {"sm_mhz", "sm_max_mhz", "reasons"}
    assert "workload" in d["config"] and "model" not in d["config"]


def _torchrun(nproc, args, timeout=900):
    port = 29600 + (os.getpid() % 1500)
    cmd = [sys.executable, "-m", "torch.distributed.run", "--nnodes=1", f"--nproc-per-node={nproc}", "--master-addr", "127.0.0.1",
           "--master-port", str(port), os.path.join(ROOT, "bench.py"), "--gpus", str(nproc)] + args
    res = subprocess.run(cmd, capture_output=True, text=True, timeout=timeout, cwd=ROOT)
    assert res.returncode == 0, res.stderr[-3000:]
    lines = [l for l in res.stdout.splitlines() if l.strip().startswith("{")]
    assert len(lines) == 1, f"exactly one JSON line expected from rank 0, got {len(lines)}"
    return json.loads(lines[0])


@pytest.mark.gpu
def test_gpu_arm_under_torchrun():
    """The N > 1 launch path of the contract on the hardware there is: torchrun, NCCL process group, barrier + max over
    ranks of the device time, rank-seeded batches.  One rank per visible GPU, at most two (this pool hands out one GPU, so
    this normally runs world size 1 through the same code: NCCL init is skipped only by torch when world == 1 is not
    launched through torchrun, never here)."""
    import torch
    n = min(torch.cuda.device_count(), 2)
    d = _torchrun(n, ["--steps", "3", "--warmup", "3", "--events", "600", "--no-cpu-baseline"])
    assert d["n_gpus"] == n and d["scaling"] == "weak" and d["value"] > 0
    assert d["config"]["events_per_gpu"] == 600
    # whole-job aggregate: the units all ranks processed over the max-over-ranks time
    assert abs(d["value"] - n * 600 / (d["ms_per_step"] * 1e-3)) / d["value"] < 1e-6
    assert d["e2e"]["value"] > 0 and d["gpu_launches"] == 4 * 3
