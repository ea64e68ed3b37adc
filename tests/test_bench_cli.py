"""bench.py contract: one JSON line with the keys the driver reads.  The reference arm (CPU oracle) runs anywhere,
also under torchrun with 2 ranks (rank 0 prints, the others exit 0 without work); the GPU arm is -m gpu."""
import json
import os
import subprocess
import sys

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
BASE_KEYS = {"metric", "value", "unit", "n_gpus", "steps", "warmup", "ms_per_step", "higher_is_better", "scaling",
             "vs_baseline", "dtype", "data", "config", "e2e", "gpu_launches", "cpu_baseline"}


def run(cmd, timeout=600):
    r = subprocess.run(cmd, cwd=ROOT, capture_output=True, text=True, timeout=timeout)
    assert r.returncode == 0, r.stderr[-2000:]
    lines = [ln for ln in r.stdout.splitlines() if ln.startswith("{")]
    return lines


def test_reference_arm_single_process():
    lines = run([sys.executable, "bench.py", "--impl", "reference", "--size", "192", "--steps", "1", "--warmup", "0"])
    assert len(lines) == 1
    d = json.loads(lines[0])
    assert BASE_KEYS <= set(d) and d["impl"] == "reference" and d["value"] > 0
    assert d["cpu_baseline"]["kind"] == "oracle" and d["cpu_baseline"]["cores"] >= 1
    assert d["e2e"]["h2d_bytes_per_step"] == 0 and d["e2e"]["d2h_bytes_per_step"] == 0 and d["e2e"]["value"] == d["value"]
    assert d["vs_baseline"] is None and d["config"]["workload"].startswith("BASELINE configs[2]")


def test_reference_arm_two_ranks_rank0_prints_once():
    cmd = [sys.executable, "-m", "torch.distributed.run", "--nnodes=1", "--nproc-per-node", "2", "--master-addr", "127.0.0.1",
           "--master-port", "29617", "bench.py", "--impl", "reference", "--gpus", "2", "--size", "160", "--steps", "1",
           "--warmup", "0"]
    lines = run(cmd)
    assert len(lines) == 1
    d = json.loads(lines[0])
    assert d["impl"] == "reference" and d["n_gpus"] == 2


@pytest.mark.gpu
def test_gpu_arm_json_line():
    lines = run([sys.executable, "bench.py", "--size", "1024", "--steps", "4", "--warmup", "3"])
    assert len(lines) == 1
    d = json.loads(lines[0])
    assert BASE_KEYS | {"roofline", "clocks", "stages", "path"} <= set(d)
    assert d["gpu_launches"] == 4 * 8 and d["steps"] == 4 and d["warmup"] >= 3
    r = d["roofline"]
    assert r["bound"] == "tensor" and r["unit"] == "TFLOP/s" and abs(r["frac"] - r["achieved"] / r["peak"]) < 1e-9
    assert d["e2e"]["h2d_bytes_per_step"] == 2 * 8 * 1024 * 1024 and d["e2e"]["matches_device_path"] is True
    assert d["cpu_baseline"]["gpu_slab_bit_exact_vs_oracle"] is True
    assert "sm_mhz" in d["clocks"] and "reasons" in d["clocks"]


@pytest.mark.gpu
def test_gpu_arm_default_run_carries_the_moduli_sweep():
    # the default workload (configs[2], N = 16) also times the config's other moduli counts; the legs after the sweep still
    # see the headline N's result
    lines = run([sys.executable, "bench.py", "--steps", "3", "--warmup", "3", "--skip-ceiling", "--skip-cpu-baseline"], timeout=900)
    d = json.loads(lines[0])
    sw = d["sweep"]
    assert [r["moduli"] for r in sw] == [14, 15, 16, 17, 18] and d["config"]["moduli"] == 16
    for r in sw:
        assert r["ms_per_step"] > 0 and 0 < r["path_frac"] < 1.2 and set(r["stage_ms"]) == {"S1", "S2", "S3", "S4S5"}
    assert d["e2e"]["matches_device_path"] is True
    assert d["roofline"]["kernel"].startswith("k3_residue_gemm_pair")
    assert d["gpu_launches"] == 3 * 8
