"""N > 1 host logic on CPU (gloo, world_size 2): DESIGN.md "Multi-GPU" is replicas only, so the one piece of
multi-rank logic is bench.py's aggregation -- job time = MAX over ranks, job units = SUM over ranks -- and the
reference arm's "rank 0 alone prints" rule.  No GPU, no oracle arithmetic."""
import json
import os
import re
import socket
import subprocess
import sys

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))

WORKER = r"""
import json, os, sys
sys.path.insert(0, {root!r})
import torch.distributed as dist
import bench
dist.init_process_group(backend="gloo")
rank, world = dist.get_rank(), dist.get_world_size()
bench.barrier()
ms, units = bench.aggregate_over_ranks(10.0 + 5.0 * rank, 1000.0 * (rank + 1))
bench.barrier()
print(json.dumps({{"rank": rank, "world": world, "ms": ms, "units": units}}), flush=True)
dist.destroy_process_group()
"""


def _free_port():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def _torchrun(nproc, argv, timeout=300):
    cmd = [sys.executable, "-m", "torch.distributed.run", "--nnodes=1", f"--nproc-per-node={nproc}",
           "--master-addr", "127.0.0.1", "--master-port", str(_free_port())] + argv
    env = dict(os.environ, OMP_NUM_THREADS="1")
    return subprocess.run(cmd, cwd=ROOT, env=env, capture_output=True, text=True, timeout=timeout)


def test_aggregate_is_max_time_sum_units_world2(tmp_path):
    script = tmp_path / "worker.py"
    script.write_text(WORKER.format(root=ROOT))
    r = _torchrun(2, [str(script)])
    assert r.returncode == 0, r.stderr[-2000:]
    rows = [json.loads(m) for m in re.findall(r"\{[^{}]*\}", r.stdout)]   # the two ranks may share a line
    assert sorted(x["rank"] for x in rows) == [0, 1]
    for x in rows:
        assert x["world"] == 2
        assert x["ms"] == 15.0          # max(10, 15)
        assert x["units"] == 3000.0     # 1000 + 2000


def test_aggregate_single_process_is_identity():
    sys.path.insert(0, ROOT)
    import bench
    assert bench.aggregate_over_ranks(3.5, 7.0) == (3.5, 7.0)


def test_reference_arm_prints_once_under_two_ranks():
    r = _torchrun(2, ["bench.py", "--impl", "reference", "--gpus", "2", "--steps", "1", "--warmup", "0", "--config", "1"])
    assert r.returncode == 0, r.stderr[-2000:]
    lines = [json.loads(ln) for ln in r.stdout.splitlines() if ln.startswith("{")]
    assert len(lines) == 1
    out = lines[0]
    assert out["impl"] == "reference" and out["n_gpus"] == 2 and out["gpu_launches"] == 0
    assert out["cpu_baseline"]["kind"] == "oracle" and out["e2e"]["h2d_bytes_per_step"] == 0
    assert out["value"] > 0
