"""World-size-2 checks of the N > 1 path on CPU (gloo).  DESIGN.md "Multi-GPU": replicas only — no data-path
collective; the only cross-rank operation is the max-over-ranks of the timed region, and under
`--impl reference` rank 0 alone works and prints."""
import json
import os
import re
import socket
import subprocess
import sys

import numpy as np

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))

WORKER = r"""
import os, sys, json
sys.path.insert(0, os.environ["ETICS_ROOT"])
import numpy as np
import torch.distributed as dist
import bench
from paper_1406_4254_b200 import workloads as W
dist.init_process_group("gloo")
rank, world = dist.get_rank(), dist.get_world_size()
ms = 10.0 + 5.0 * rank                       # the slower rank decides
mx = bench.max_over_ranks(ms, "cpu")
pos, mass = W.particles("hernquist", 64, seed=bench.replica_seed(rank))
print("RESULT " + json.dumps({"rank": rank, "world": world, "max_ms": mx,
      "value": bench.whole_job_value(world, 1000, mx), "x0": float(pos[0, 0])}), flush=True)
dist.destroy_process_group()
"""


def _free_port():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def _torchrun(args, extra_env=None, timeout=300):
    env = dict(os.environ, ETICS_ROOT=ROOT, OMP_NUM_THREADS="2")
    env.update(extra_env or {})
    cmd = [sys.executable, "-m", "torch.distributed.run", "--nnodes=1", "--nproc-per-node", "2",
           "--master-addr", "127.0.0.1", "--master-port", str(_free_port())] + args
    return subprocess.run(cmd, capture_output=True, text=True, timeout=timeout, env=env, cwd=ROOT)


def test_max_over_ranks_and_replica_seeds(tmp_path):
    w = tmp_path / "worker.py"
    w.write_text(WORKER)
    r = _torchrun([str(w)])
    assert r.returncode == 0, r.stderr[-2000:]
    # the two ranks share one stdout: their lines may run together, so pick the records out by pattern
    res = [json.loads(m) for m in re.findall(r"RESULT (\{[^{}]*\})", r.stdout)]
    assert sorted(x["rank"] for x in res) == [0, 1]
    for x in res:
        assert x["world"] == 2
        assert x["max_ms"] == 15.0                      # max over ranks, on every rank
        assert np.isclose(x["value"], 2 * 1000 / 15e-3)    # whole-job aggregate: both replicas' particles
    assert res[0]["x0"] != res[1]["x0"]                 # each replica has its own particle set


def test_reference_arm_only_rank0_prints():
    r = _torchrun(["bench.py", "--impl", "reference", "--gpus", "2", "--steps", "1", "--warmup", "0", "--ref-budget", "1"])
    assert r.returncode == 0, r.stderr[-2000:]
    lines = [l for l in r.stdout.splitlines() if l.startswith("{")]
    assert len(lines) == 1
    d = json.loads(lines[0])
    assert d["impl"] == "reference" and d["n_gpus"] == 2 and d["gpu_launches"] == 0
    assert d["cpu_baseline"]["kind"] == "oracle" and d["e2e"]["h2d_bytes_per_step"] == 0
    assert d["value"] > 0 and d["unit"] == "particles/s"
