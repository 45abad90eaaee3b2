"""The N > 1 path of bench.py on CPU: two processes, gloo, 127.0.0.1.  The method does not shard
(replicas only), so what the ranks share is the barrier, the MAX of their times
and the aggregate; the reference arm runs on rank 0 alone."""
import json
import os
import socket
import subprocess
import sys

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _free_port():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


WORKER = r"""
import os, sys
sys.path.insert(0, %r)
import torch.distributed as dist
import bench
dist.init_process_group("gloo", init_method="tcp://127.0.0.1:%%s" %% sys.argv[1], rank=int(sys.argv[2]), world_size=2)
rank = dist.get_rank()
dist.barrier()
ms = bench.max_over_ranks(10.0 + 5.0 * rank, dist, "cpu")      # rank 1 is the slow one
assert ms == 15.0, ms
v = bench.whole_job_value(2, 300, ms)
assert abs(v - 2 * 300 / 15e-3) < 1e-9
assert bench.max_over_ranks(3.0, None, "cpu") == 3.0
dist.barrier()
dist.destroy_process_group()
print("ok", rank)
""" % ROOT


def test_max_over_ranks_and_aggregate_gloo_world2(tmp_path):
    port = _free_port()
    script = tmp_path / "worker.py"
    script.write_text(WORKER)
    procs = [subprocess.Popen([sys.executable, str(script), str(port), str(r)], stdout=subprocess.PIPE, stderr=subprocess.PIPE,
                              text=True) for r in range(2)]
    outs = [p.communicate(timeout=120) for p in procs]
    for r, (p, (o, e)) in enumerate(zip(procs, outs)):
        assert p.returncode == 0, e[-2000:]
        assert o.strip().endswith(f"ok {r}")


def test_reference_arm_runs_on_rank0_only():
    env = dict(os.environ, RANK="1", WORLD_SIZE="2", LOCAL_RANK="1")
    out = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--impl", "reference", "--config", "lj_1k", "--steps", "3",
                          "--warmup", "3", "--gpus", "2"], env=env, capture_output=True, text=True, timeout=300)
    assert out.returncode == 0 and out.stdout.strip() == ""
    env["RANK"] = "0"
    out = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--impl", "reference", "--config", "lj_1k", "--steps", "3",
                          "--warmup", "3", "--gpus", "2"], env=env, capture_output=True, text=True, timeout=300)
    assert out.returncode == 0, out.stderr[-2000:]
    line = json.loads(out.stdout.strip().splitlines()[-1])
    assert line["impl"] == "reference" and line["value"] > 0 and line["cpu_baseline"]["kind"] == "oracle"
    assert line["e2e"]["h2d_bytes_per_step"] == 0 and line["n_gpus"] == 2
