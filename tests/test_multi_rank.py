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


SHARD_WORKER = r"""
import os, sys, json
sys.path.insert(0, os.environ["ETICS_ROOT"])
import numpy as np
import torch, torch.distributed as dist
import oracle
from paper_1406_4254_b200 import sharded, workloads as W
dist.init_process_group("gloo")
rank, world = dist.get_rank(), dist.get_world_size()
n, nmax, lmax = 2001, 6, 4
pos, mass = W.particles("hernquist", n, seed=4, axes=(1.0, 0.8, 0.6))
a, b = sharded.shard_range(n, rank, world)
# the exchange logic of sharded.scf_force_sharded, with the oracle standing in for the kernels (no GPU here):
A, B = oracle.scf_coeffs(np.ascontiguousarray(pos[:, a:b]), mass[a:b], nmax, lmax)
local = torch.from_numpy(np.concatenate([A, B]))
def all_gather(t):
    stack = [torch.empty_like(t) for _ in range(world)]
    dist.all_gather(stack, t)
    return torch.stack(stack)
def combine(stack):
    s = stack[0].clone()
    for r in range(1, stack.shape[0]):
        s += stack[r]
    return s
table = sharded.gather_and_combine(local, all_gather, combine).numpy()
T = len(A)
acc, pot = oracle.scf_force(np.ascontiguousarray(pos[:, a:b]), nmax, lmax, table[:T], table[T:])
A0, B0 = oracle.scf_coeffs(pos, mass, nmax, lmax)
acc0, pot0 = oracle.scf_force(pos, nmax, lmax, A0, B0)
print("RESULT " + json.dumps({"rank": rank, "first": a, "last": b,
      "errA": float(np.max(np.abs(table[:T] - A0)) / np.max(np.abs(A0))),
      "errpot": float(np.max(np.abs(pot - pot0[a:b]) / np.abs(pot0[a:b]))),
      "digest": float(np.sum(table * np.arange(1, 2 * T + 1)))}), flush=True)
dist.destroy_process_group()
"""


def test_shard_ranges_cover_every_particle_once():
    from paper_1406_4254_b200 import sharded
    for n in (0, 1, 7, 1000, 1001, 12345):
        for world in (1, 2, 3, 8):
            r = [sharded.shard_range(n, k, world) for k in range(world)]
            assert r[0][0] == 0 and r[-1][1] == n
            assert all(r[k][1] == r[k + 1][0] for k in range(world - 1))
            sizes = [b - a for a, b in r]
            assert max(sizes) - min(sizes) <= 1


def test_sharded_scf_exchange_two_ranks(tmp_path):
    """SURVEY 8(f)3 / PAPER.md:195, :221: coefficients of the shards, gathered and added in rank order, are the coefficients
    of the whole set (to summation rounding), identical on both ranks; every rank's shard then gets the whole set's field."""
    w = tmp_path / "shard_worker.py"
    w.write_text(SHARD_WORKER)
    r = _torchrun([str(w)])
    assert r.returncode == 0, r.stderr[-2000:]
    res = sorted((json.loads(m) for m in re.findall(r"RESULT (\{[^{}]*\})", r.stdout)), key=lambda x: x["rank"])
    assert [x["rank"] for x in res] == [0, 1]
    assert res[0]["first"] == 0 and res[0]["last"] == res[1]["first"] and res[1]["last"] == 2001
    for x in res:
        assert x["errA"] < 1e-13 and x["errpot"] < 1e-12
    assert res[0]["digest"] == res[1]["digest"]          # bit-identical tables on both ranks


MEX_SHARD_WORKER = r"""
import os, sys, json
sys.path.insert(0, os.environ["ETICS_ROOT"])
import numpy as np
import torch, torch.distributed as dist
import oracle
from paper_1406_4254_b200 import sharded, workloads as W
dist.init_process_group("gloo")
rank, world = dist.get_rank(), dist.get_world_size()
n, lmax = 3001, 4
pos, mass = W.particles("hernquist", n, seed=7)
pos = pos.copy(); mass = mass.copy()
mass *= 1.0 + 0.5 * np.sin(np.arange(n))              # unequal masses: a misrouted row cannot go unnoticed
# ties ACROSS the index shards: particles of the second half at the radius of particles of the first half (same key bits)
for j in range(0, 40):
    pos[:, n // 2 + 5 + 3 * j] = pos[[1, 0, 2], 7 * j] * np.array([-1.0, 1.0, -1.0])
a, b = sharded.shard_range(n, rank, world)
acc0, pot0, perm0 = oracle.mex_force(pos, mass, lmax, return_perm=True)     # the whole set on every rank: the expected answer
checks = {}

# stand-ins for the kernels (no GPU here); what is under test is the partition, the exchange and the return path
def sort(p):
    k, pm = oracle.mex_sort(p.numpy())
    return torch.from_numpy(k.view(np.int64)), torch.from_numpy(pm.astype(np.int32))
def moments(pos_r, mass_r):
    nr = mass_r.numel()
    return torch.tensor([float(nr), float(mass_r.sum())], dtype=torch.float64), (pos_r, mass_r)
def bases(parts, r):
    return torch.stack([parts[:r, 0].sum(), parts[r + 1:, 1].sum()])
def force(state, base):
    pos_r, mass_r = state[0].numpy(), state[1].numpy()
    nr, c0 = len(mass_r), int(base[0])
    _, pr = oracle.mex_sort(pos_r)
    want = perm0[c0:c0 + nr].astype(np.int64)           # this key range = a slice of the whole set's sorted order ...
    checks["range_is_slice"] = bool(np.array_equal(pos_r[:, pr], pos[:, want]) and np.array_equal(mass_r[pr], mass[want]))
    checks["mass_outside"] = bool(np.isclose(float(base[1]), mass[perm0[c0 + nr:].astype(np.int64)].sum(), rtol=1e-12))
    acc_r = np.empty((3, nr)); pot_r = np.empty(nr)
    acc_r[:, pr] = acc0[:, want]; pot_r[pr] = pot0[want]   # ... whose answer is known: hand it out in arrival order
    return torch.from_numpy(acc_r), torch.from_numpy(pot_r)

acc, pot = sharded.mex_force_partitioned(torch.from_numpy(np.ascontiguousarray(pos[:, a:b])), torch.from_numpy(mass[a:b].copy()),
                                         sort, moments, bases, force)
print("RESULT " + json.dumps({"rank": rank, **checks,
      "exact": bool(np.array_equal(acc.numpy(), acc0[:, a:b]) and np.array_equal(pot.numpy(), pot0[a:b]))}), flush=True)
dist.destroy_process_group()
"""


def test_radius_partition_helpers():
    import torch
    from paper_1406_4254_b200 import sharded
    assert sharded.sample_positions(1, 4) == [0, 0, 0, 0]
    assert sharded.sample_positions(8, 4) == [1, 3, 5, 7]
    keys = torch.tensor([1, 2, 2, 3, 5, 8])
    # equal keys never straddle a splitter: both 2s go to rank 1
    assert sharded.send_counts(keys, torch.tensor([2, 6])) == [1, 4, 1]
    assert sharded.send_counts(keys, torch.tensor([], dtype=torch.int64)) == [6]
    assert sharded.send_counts(keys, torch.tensor([0, 100])) == [0, 6, 0]      # empty ranges are legal
    assert sharded.choose_splitters(torch.tensor([[1, 5, 9, 13], [2, 6, 10, 14]]), 2).tolist() == [9]
    assert sharded.choose_splitters(torch.tensor([[3, 1, 2]]), 1).numel() == 0


def test_radius_partitioned_mex_exchange_two_ranks(tmp_path):
    """every rank's key range is a contiguous slice of the whole set's sorted order (ties
    across the index shards included, in global index order), the interior-count / exterior-mass bases are the sums over the
    ranks inside / outside, and every particle's result returns to its owner at its original index."""
    w = tmp_path / "mex_shard_worker.py"
    w.write_text(MEX_SHARD_WORKER)
    r = _torchrun([str(w)])
    assert r.returncode == 0, r.stderr[-2000:]
    res = sorted((json.loads(m) for m in re.findall(r"RESULT (\{[^{}]*\})", r.stdout)), key=lambda x: x["rank"])
    assert [x["rank"] for x in res] == [0, 1]
    for x in res:
        assert x["range_is_slice"] and x["mass_outside"] and x["exact"]
