"""The N > 1 path on real GPUs: template shards on two ranks over NCCL, launched
the way the driver launches bench.py.  Needs two visible GPUs; on a one-GPU box the tests are
SKIPPED, loudly -- the multi-GPU path is then covered by tests/test_shard_gloo.py (host logic)
and test_sharded_search_equals_unsharded (one GPU) only, and stays unmeasured on hardware."""
import os
import socket
import subprocess
import sys

import pytest

torch = pytest.importorskip("torch")

pytestmark = pytest.mark.gpu
ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _free_port() -> int:
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def _need_two_gpus():
    n = torch.cuda.device_count()
    if n < 2:
        pytest.skip(f"MULTI-GPU PATH NOT RUN: {n} CUDA device(s) visible, 2 needed "
                    "(torch.distributed.run --nproc-per-node 2 over NCCL)")


def _torchrun(script_args, timeout=600):
    cmd = [sys.executable, "-m", "torch.distributed.run", "--nnodes=1", "--nproc-per-node", "2",
           "--master-addr", "127.0.0.1", "--master-port", str(_free_port())] + script_args
    return subprocess.run(cmd, cwd=ROOT, capture_output=True, text=True, timeout=timeout)


def test_sharded_search_on_two_gpus_equals_unsharded_and_oracle():
    _need_two_gpus()
    r = _torchrun([os.path.join(ROOT, "tests", "dist_worker_nccl.py")])
    assert r.returncode == 0, r.stdout[-2000:] + r.stderr[-4000:]


def test_bench_on_two_gpus_prints_one_weak_scaling_line():
    """bench.py --gpus 2 as the driver runs it: one JSON line from rank 0, aggregate over both
    ranks, max-over-ranks timing (a short run: 256 templates per GPU)."""
    import json

    _need_two_gpus()
    r = _torchrun([os.path.join(ROOT, "bench.py"), "--gpus", "2", "--steps", "2", "--warmup", "3",
                   "--templates", "256", "--no-cpu-baseline", "--no-side"])
    assert r.returncode == 0, r.stdout[-2000:] + r.stderr[-4000:]
    lines = [ln for ln in r.stdout.splitlines() if ln.startswith("{")]
    assert len(lines) == 1
    d = json.loads(lines[0])
    assert d["n_gpus"] == 2 and d["scaling"] == "weak"
    assert d["value"] > 0 and d["config"]["templates_per_gpu"] == 256
