"""bench.py's N>1 branch (process group, barrier, max over ranks, shard offsets) run for real: two ranks under
torch.distributed.run with the gloo backend, both on the one GPU of this box (--device-index 0).  The data path has no
collective (contiguous index ranges), so the ranks never wait on each other's kernels; they
time-share the GPU, and the aggregate rate must come out near the single-process rate."""
import json
import os
import subprocess
import sys

import pytest
import torch

from paper_2602_05606_b200 import kappagen as kg

pytestmark = pytest.mark.gpu

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def test_two_ranks_on_one_gpu_print_one_aggregate_line():
    steps, n = 10, 1 << 28
    cmd = [sys.executable, "-m", "torch.distributed.run", "--nnodes=1", "--nproc-per-node", "2", "--master-addr", "127.0.0.1",
           "--master-port", "29533", os.path.join(ROOT, "bench.py"), "--gpus", "2", "--dist-backend", "gloo", "--device-index", "0",
           "--steps", str(steps), "--warmup", "3", "--e2e-steps", "1", "--no-extras"]
    r = subprocess.run(cmd, capture_output=True, text=True, timeout=900, cwd=ROOT)
    assert r.returncode == 0, r.stderr[-3000:]
    lines = [l for l in r.stdout.splitlines() if l.startswith("{")]
    assert len(lines) == 1, r.stdout                                   # rank 0 alone prints
    line = json.loads(lines[0])
    assert line["n_gpus"] == 2 and line["scaling"] == "weak" and "x2" in line["config"]["parallelism"]
    assert line["config"]["dist_backend"] == "gloo" and line["steps"] == steps and "extras" not in line
    assert line["e2e"]["d2h_bytes_per_step"] == 2 * 12 * n
    # each rank owns the index range [(s*2 + r) * 2^28, +2^28) of step s: its last step, recomputed here
    assert [s["rank"] for s in line["shards"]] == [0, 1]
    for s in line["shards"]:
        assert s["offset"] == ((steps - 1) * 2 + s["rank"]) * n
        vx = kg.sample(4, 2.0, 0.1, 42, s["offset"], "f32")[0]
        assert [float(v) for v in vx.double().cpu()] == s["vx_head"]
    # two processes time-share one GPU: the aggregate stays near what one process reaches alone
    planes = tuple(torch.empty(n, dtype=torch.float32, device="cuda") for _ in range(3))
    for s in range(3):
        kg.sample(n, 2.0, 0.1, 42, s * n, "f32", out=planes)
    a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    a.record()
    for s in range(steps):
        kg.sample(n, 2.0, 0.1, 42, s * n, "f32", out=planes)
    b.record()
    torch.cuda.synchronize()
    alone = steps * n / (a.elapsed_time(b) * 1e-3)
    assert 0.6 <= line["value"] / alone <= 1.15, (line["value"], alone)
