"""Multi-GPU spin sharding on the CUDA path (SURVEY.md 8(e) / 8(f) f3; PAPER.md:116 spin independence, :194 signals
added afterwards, :374 "not yet tested in a multi-GPU system").

`bench.py --scaling strong` is the code path a scaling run takes: every rank builds the SAME named workload, keeps the
contiguous spin range `dist.shard_bounds` gives it, simulates its shard through the C-ABI, and ONE collective adds the
per-rank signals in rank order; rank 0 then checks the reduced signal against the 1-GPU signal of the whole workload
(5e-6 of its maximum).  The 2-rank NCCL test needs two GPUs and is skipped on the 1-GPU boxes of this project; the
1-rank run of the same arm and the host-side sharding are always exercised."""
import json
import os
import socket
import subprocess
import sys

import numpy as np
import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _free_port():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def _last_json(text):
    for line in reversed(text.strip().splitlines()):
        if line.startswith("{"):
            return json.loads(line)
    raise AssertionError("no JSON line in the bench output:\n" + text[-2000:])


def test_strong_scaling_shards_partition_the_named_workload():
    """Host side of the strong-scaling arm: the shards of the ranks are disjoint, contiguous, and together the workload."""
    sys.path.insert(0, ROOT)
    import bench
    for world in (1, 2, 3, 8):
        parts = [bench.make_workload("1", r, world, "strong") for r in range(world)]
        whole = parts[0][1]
        for k in ("x", "y", "z", "M0", "T1", "T2", "dw"):
            assert np.array_equal(np.concatenate([getattr(p[0].phantom, k) for p in parts]), getattr(whole.phantom, k))
        sizes = [p[0].phantom.n for p in parts]
        assert max(sizes) - min(sizes) <= 1 and sum(sizes) == whole.phantom.n
        for p in parts:                                        # the plan is replicated: every rank builds the same sequence
            assert p[0].seq is p[1].seq and np.array_equal(p[0].seq.adc_t, whole.seq.adc_t) and \
                np.array_equal(p[0].seq.rf_re, whole.seq.rf_re)


@pytest.mark.gpu
def test_strong_scaling_arm_on_one_gpu_is_the_plain_run():
    import torch
    if not torch.cuda.is_available():
        pytest.skip("no CUDA device")
    cmd = [sys.executable, os.path.join(ROOT, "bench.py"), "--gpus", "1", "--steps", "2", "--warmup", "3", "--workload", "2",
           "--extra", "none", "--no-cpu-baseline"]
    strong = _last_json(subprocess.run(cmd + ["--scaling", "strong"], capture_output=True, text=True, check=True,
                                       cwd=ROOT).stdout)
    weak = _last_json(subprocess.run(cmd, capture_output=True, text=True, check=True, cwd=ROOT).stdout)
    assert strong["scaling"] == "strong" and strong["shard_check"]["ok"] and strong["shard_check"]["max_err_vs_1gpu"] == 0.0
    for k in ("workload", "n_spins_total", "n_intervals", "spin_steps_per_step", "path"):
        assert strong["config"][k] == weak["config"][k]
    assert strong["gpu_launches"] == weak["gpu_launches"] > 0
    assert 0.5 < strong["value"] / weak["value"] < 2.0          # the same computation, timed twice


@pytest.mark.gpu
def test_two_nccl_ranks_shard_config2_and_reduce_to_the_one_gpu_signal():
    import torch
    if not torch.cuda.is_available() or torch.cuda.device_count() < 2:
        pytest.skip("needs 2 GPUs (the boxes of this project have one); the 1-rank arm and the gloo tests cover the rest")
    env = dict(os.environ, NCCL_DEBUG="INFO")     # the communicator lines are evidence that NCCL carried the sum
    cmd = [sys.executable, "-m", "torch.distributed.run", "--nnodes=1", "--nproc-per-node", "2", "--master-addr",
           "127.0.0.1", "--master-port", str(_free_port()), os.path.join(ROOT, "bench.py"), "--gpus", "2", "--steps", "2",
           "--warmup", "3", "--workload", "2", "--scaling", "strong", "--extra", "none", "--no-cpu-baseline"]
    res = subprocess.run(cmd, capture_output=True, text=True, cwd=ROOT, env=env, timeout=600)
    assert res.returncode == 0, res.stderr[-3000:]
    out = _last_json(res.stdout)
    assert out["n_gpus"] == 2 and out["scaling"] == "strong" and out["shard_check"]["ok"]
    assert out["config"]["n_spins_per_gpu"] * 2 == out["config"]["n_spins_total"] == 16384
    assert "NCCL INFO" in res.stdout + res.stderr
