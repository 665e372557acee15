"""N > 1 is "replicas only": no data-path collective. What crosses ranks is the bench's
max-over-ranks of the step time and the rank-0-only reporting. Covered here with world-size-2 gloo on the CPU."""
import json
import os
import socket
import subprocess
import sys

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _free_port() -> int:
    s = socket.socket()
    s.bind(("127.0.0.1", 0))
    p = s.getsockname()[1]
    s.close()
    return p


def _torchrun(args, attempts=2):
    """World-size-2 launch on 127.0.0.1; a rendezvous that loses the race for its port is retried on a new one."""
    env = dict(os.environ, OMP_NUM_THREADS="2")
    for _ in range(attempts):
        cmd = [sys.executable, "-m", "torch.distributed.run", "--nnodes=1", "--nproc-per-node", "2",
               "--master-addr", "127.0.0.1", "--master-port", str(_free_port())] + list(args)
        r = subprocess.run(cmd, capture_output=True, text=True, timeout=900, cwd=ROOT, env=env)
        if r.returncode == 0:
            break
    return r


_WORKER = r"""
import os, sys, json
sys.path.insert(0, {root!r})
import torch.distributed as dist
import bench
dist.init_process_group("gloo")
r, w = dist.get_rank(), dist.get_world_size()
local_ms = 10.0 + 5.0 * r                      # rank 1 is the slow replica
ms = bench.max_over_ranks(local_ms, dist, "cpu")
v = bench.whole_job_value(w, 1000.0, 4, ms * 1e-3)
for turn in range(w):                          # one rank prints at a time: two ranks writing to the one pipe at the
    dist.barrier()                             # same moment can interleave within a line
    if turn == r:
        sys.stdout.write(json.dumps({{"rank": r, "world": w, "ms": ms, "value": v}}) + "\n")
        sys.stdout.flush()
dist.barrier()
dist.destroy_process_group()
"""


def test_max_over_ranks_and_whole_job_value_world2(tmp_path):
    script = tmp_path / "worker.py"
    script.write_text(_WORKER.format(root=ROOT))
    r = _torchrun([str(script)])
    assert r.returncode == 0, r.stderr[-2000:]
    lines = [json.loads(l) for l in r.stdout.splitlines() if l.startswith("{")]
    assert sorted(l["rank"] for l in lines) == [0, 1]
    for l in lines:
        assert l["world"] == 2
        assert l["ms"] == 15.0                                  # the max, on every rank
        assert l["value"] == pytest.approx(2 * 1000.0 * 4 / 15e-3)  # both replicas' work over the slowest time


def test_reference_arm_under_torchrun_prints_one_line_from_rank0():
    """bench.py --impl reference with N = 2: rank 0 alone runs the oracle and prints; rank 1 exits 0 silently."""
    r = _torchrun([os.path.join(ROOT, "bench.py"), "--impl", "reference", "--gpus", "2", "--steps", "1",
                   "--warmup", "0", "--config", "1"])
    assert r.returncode == 0, r.stderr[-2000:]
    lines = [json.loads(l) for l in r.stdout.splitlines() if l.startswith("{")]
    assert len(lines) == 1
    d = lines[0]
    assert d["impl"] == "reference" and d["n_gpus"] == 2 and d["unit"] == "updates/s"
    assert d["cpu_baseline"]["kind"] == "oracle" and d["cpu_baseline"]["cores"] >= 1
    assert d["e2e"]["h2d_bytes_per_step"] == 0 and d["e2e"]["value"] == d["value"] > 0


def test_single_process_helpers_without_dist():
    sys.path.insert(0, ROOT)
    import bench
    assert bench.max_over_ranks(3.5, None, "cpu") == 3.5
    assert bench.whole_job_value(1, 10.0, 2, 0.5) == 40.0
