"""-m gpu smoke of bench.py's N > 1 arm: two ranks (sharing this box's one GPU, gradients exchanged over gloo) run the
sharded step of DESIGN.md section 10 -- same model on every rank, brick slabs / point slices, global loss normaliser, one
all-reduce on the flat gradient buffer.  It proves the code path runs and prints a well-formed line; it is not a measurement
(NCCL needs one GPU per rank; the driver's scaling runs use it)."""
import json
import os
import subprocess
import sys

import pytest

pytestmark = pytest.mark.gpu
ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.mark.parametrize("workload", ["c1"])
def test_two_ranks_over_gloo(workload):
    env = dict(os.environ, GS_BENCH_BACKEND="gloo")
    cmd = [sys.executable, "-m", "torch.distributed.run", "--nnodes=1", "--nproc-per-node", "2", "--master-addr", "127.0.0.1",
           "--master-port", "29533", os.path.join(ROOT, "bench.py"), "--gpus", "2", "--steps", "3", "--warmup", "3", "--workload", workload,
           "--no-cpu"]
    r = subprocess.run(cmd, cwd=ROOT, env=env, capture_output=True, text=True, timeout=600)
    assert r.returncode == 0, r.stderr[-2000:]
    lines = [l for l in r.stdout.splitlines() if l.startswith("{")]
    assert len(lines) == 1          # rank 0 alone prints
    d = json.loads(lines[0])
    assert d["n_gpus"] == 2 and d["scaling"] == "strong" and d["value"] > 0 and d["gpu_launches"] > 0
    assert d["config"]["points_per_step"] == 32 ** 3   # the whole grid, split over the ranks
