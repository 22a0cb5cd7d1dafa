"""bench.py without a GPU: algorithmic-work helpers against BASELINE.md's table, the reference arm
(the oracle on the host cores, same metric / config object as the GPU arm), and `--gpus N` refusing
to pretend when the box has fewer than N devices."""
import json
import os
import subprocess
import sys

import pytest
import torch

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
sys.path.insert(0, ROOT)

import bench  # noqa: E402
import ttt_inputs as ti  # noqa: E402


def test_algorithmic_flops_and_bytes_match_baseline_md():
    # GFLOP per chunk (18 M d H [+ NS]) and algorithmic HBM MB per chunk
    for name, gflop, ns_gflop, mb in (("cfg2", 25.93, 0.0, 90.7), ("cfg3", 51.87, 1.13, 90.7),
                                      ("cfg4", 207.47, 0.0, 363.0), ("cfg5", 413.88, 4.53, 360.7)):
        w = ti.CONFIGS[name]
        M = w.chunk_tokens
        assert abs(18.0 * M * w.d * w.hidden / 1e9 - gflop) < 0.01 * gflop
        assert abs(bench.flops_per_chunk(w, M, "step") / 1e9 - (gflop + ns_gflop)) < 0.01 * gflop
        assert abs(bench.flops_per_chunk(w, M, "update") + bench.flops_per_chunk(w, M, "apply")
                   - bench.flops_per_chunk(w, M, "step")) < 1.0
        assert abs(bench.bytes_per_chunk(w, M) / 1e6 - mb) < 0.01 * mb
    # the paper's shape: 18 * 82440 * 1024 * 4096 = 6.22 TFLOP per chunk
    w = ti.CONFIGS["paper_k4"]
    assert abs(bench.flops_per_chunk(w, w.chunk_tokens) / 1e12 - 6.22) < 0.01
    for name in bench.PERF_WORKLOADS:
        w = ti.CONFIGS[name]
        assert bench.n_input_sets(w) * bench.bytes_per_chunk(w, w.chunk_tokens) > 2 * bench.L2_BYTES


def test_reference_arm_prints_the_contract_line():
    r = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--impl", "reference", "--workload",
                        "cfg2", "--steps", "1", "--warmup", "0"], capture_output=True, text=True, timeout=300,
                       cwd=ROOT)
    assert r.returncode == 0, r.stderr[-2000:]
    line = json.loads(r.stdout.strip().splitlines()[-1])
    assert line["impl"] == "reference" and line["metric"] == "ttt_update_apply_tokens_per_s"
    assert line["unit"] == "tokens/s" and line["higher_is_better"] is True and line["value"] > 0
    assert line["config"] == bench.config_of(ti.CONFIGS["cfg2"], 1)        # the GPU arm prints the same object
    assert line["cpu_baseline"]["kind"] == "oracle" and line["cpu_baseline"]["cores"] >= 1
    assert line["e2e"]["h2d_bytes_per_step"] == 0 and line["gpu_launches"] == 0


@pytest.mark.skipif(torch.cuda.device_count() >= 2, reason="needs a box with fewer than 2 GPUs")
def test_gpus_flag_fails_loudly_without_enough_devices():
    env = {k: v for k, v in os.environ.items() if k not in ("WORLD_SIZE", "RANK", "LOCAL_RANK")}
    r = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--gpus", "2", "--steps", "1"],
                       capture_output=True, text=True, timeout=300, cwd=ROOT, env=env)
    assert r.returncode != 0
    assert "--gpus 2" in r.stderr and "CUDA device" in r.stderr
    assert "n_gpus" not in r.stdout
