"""Radius-partitioned MEX on ONE GPU: the shards of a radius partition are run
one after the other through etics_mex_shard_moments / _bases / _force and must reproduce the oracle's MEX of the whole set
(1e-10, tests/parity.py).  The exchange between ranks is covered on CPU (tests/test_multi_rank.py, gloo, world size 2)."""
import os
import subprocess
import sys

import numpy as np
import pytest

import oracle
from paper_1406_4254_b200 import workloads as W
from parity import TOL, rel_err_scalar, rel_err_vector

torch = pytest.importorskip("torch")
pytestmark = pytest.mark.gpu
ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def E():
    assert torch.cuda.is_available(), "GPU tests need a CUDA device"
    from paper_1406_4254_b200 import binding
    binding.lib()
    binding.etics_init()
    return binding


def dev(a):
    return torch.from_numpy(np.ascontiguousarray(a)).cuda()


def workspace(E, n, lmax):
    return torch.empty(E.etics_workspace_bytes(E.ETICS_WS_MEX_FORCE, n, 0, lmax), dtype=torch.uint8, device="cuda")


def particle_set(n, seed):
    pos, mass = W.particles("hernquist", n, seed=seed, axes=(1.0, 0.8, 0.6))
    pos, mass = pos.copy(), mass.copy()
    mass *= 1.0 + 0.5 * np.sin(np.arange(n))
    for j in range(min(50, n // 4)):                                  # equal radii at distant indices
        pos[:, n // 2 + 2 * j] = pos[[2, 0, 1], 3 * j] * np.array([1.0, -1.0, -1.0])
    pos[:, 5] = [0.0, 0.0, 0.37]                                        # on the z axis
    return pos, mass


def radius_shards(pos, cuts):
    """Index sets of a radius partition: cut positions in the sorted order, moved so that equal keys stay together; inside a
    shard the particles keep the order of their indices."""
    keys, perm = oracle.mex_sort(pos)
    n = len(perm)
    edges = [0]
    for c in cuts:
        c = min(max(int(c), 0), n)
        while 0 < c < n and keys[c] == keys[c - 1]:
            c += 1
        edges.append(max(c, edges[-1]))
    edges.append(n)
    return [np.sort(perm[a:b].astype(np.int64)) for a, b in zip(edges[:-1], edges[1:])]


def run_shards(E, pos, mass, lmax, shards, what=None):
    what = E.ETICS_WHAT_BOTH if what is None else what
    R = E.etics_mex_shard_rows(lmax)
    parts = torch.zeros((len(shards), R), dtype=torch.float64, device="cuda")
    state = []
    for s, idx in enumerate(shards):
        if len(idx) == 0:
            state.append(None)
            continue
        ws = workspace(E, len(idx), lmax)
        E.etics_mex_shard_moments(dev(pos[:, idx]), dev(mass[idx]), lmax, ws, totals=parts[s])
        state.append(ws)
    acc = np.full((3, len(mass)), np.nan)
    pot = np.full(len(mass), np.nan)
    for s, idx in enumerate(shards):
        if len(idx) == 0:
            continue
        base = E.etics_mex_shard_bases(parts, s, lmax)
        a, p = E.etics_mex_shard_force(len(idx), lmax, what, base, state[s])
        torch.cuda.synchronize()
        if a is not None:
            acc[:, idx] = a.cpu().numpy()
        if p is not None:
            pot[idx] = p.cpu().numpy()
    return acc, pot


@pytest.mark.parametrize("lmax", [0, 1, 6, 8, 10])
def test_one_shard_has_the_bits_of_mex_force(E, lmax):
    pos, mass = particle_set(5000 + lmax, seed=20 + lmax)
    acc, pot = run_shards(E, pos, mass, lmax, [np.arange(len(mass))])
    a0, p0 = E.etics_mex_force(dev(pos), dev(mass), lmax)
    torch.cuda.synchronize()
    assert np.array_equal(acc, a0.cpu().numpy()) and np.array_equal(pot, p0.cpu().numpy())


@pytest.mark.parametrize("lmax,n,cuts", [
    (6, 20011, [10000]),                         # two halves
    (6, 20011, [1, 300, 4096, 4097, 19000]),     # a one-particle innermost shard, cuts at and next to a sort-tile boundary
    (2, 777, [0, 400, 777]),                     # empty shards at both ends
    (0, 3001, [1000, 2000]),
    (8, 30011, [7000, 7001, 22000]),             # a one-particle shard in the middle
    (10, 9001, [3000, 6000]),
])
def test_radius_shards_match_the_oracle(E, lmax, n, cuts):
    pos, mass = particle_set(n, seed=31 + lmax)
    shards = radius_shards(pos, cuts)
    assert sum(len(s) for s in shards) == n
    acc, pot = run_shards(E, pos, mass, lmax, shards)
    acc0, pot0 = oracle.mex_force(pos, mass, lmax)
    assert rel_err_scalar(pot, pot0, floor=0.0) <= TOL
    assert rel_err_vector(acc, acc0) <= TOL


def test_config3_full_size_in_four_radius_shards(E):
    """BASELINE.json configs[2] (N = 10^6 Hernquist sphere, lmax = 6) split into four radius ranges of unequal size: the shards
    of a 4-GPU run, one after the other on this GPU, against the oracle's MEX of the whole set."""
    pos, mass = W.config_particles(3)
    n = len(mass)
    shards = radius_shards(pos, [n // 5, n // 2, n - 4097])
    acc, pot = run_shards(E, pos, mass, 6, shards)
    acc0, pot0 = oracle.mex_force(pos, mass, 6)
    assert rel_err_scalar(pot, pot0, floor=0.0) <= TOL
    assert rel_err_vector(acc, acc0) <= TOL


def test_shard_variants_and_determinism(E):
    lmax = 5
    pos, mass = particle_set(12007, seed=3)
    shards = radius_shards(pos, [2500, 9000])
    acc, pot = run_shards(E, pos, mass, lmax, shards)
    acc2, pot2 = run_shards(E, pos, mass, lmax, shards)
    assert np.array_equal(acc, acc2) and np.array_equal(pot, pot2)             # fixed summation order everywhere
    _, potp = run_shards(E, pos, mass, lmax, shards, E.ETICS_WHAT_POTENTIAL)
    accf, _ = run_shards(E, pos, mass, lmax, shards, E.ETICS_WHAT_FORCE)
    assert np.array_equal(accf, acc)                                           # force only = 'both' without the store of Phi
    assert rel_err_scalar(potp, pot, floor=0.0) <= 1e-14                       # its own kernel instance: rounding order only


def test_shard_bases_are_ordered_sums(E):
    lmax, nparts = 4, 5
    R = E.etics_mex_shard_rows(lmax)
    rng = np.random.default_rng(5)
    parts = rng.standard_normal((nparts, R)) * 10.0 ** rng.integers(-8, 8, size=(nparts, R))
    n_in = n_out = 0
    for rank in range(nparts):
        base = E.etics_mex_shard_bases(dev(parts), rank, lmax).cpu().numpy()
        inner = np.zeros(R)
        for s in range(rank):                       # from the innermost shard outwards
            inner = inner + parts[s]
        outer = np.zeros(R)
        for s in range(nparts - 1, rank, -1):       # from the outermost shard inwards
            outer = outer + parts[s]
        is_in, is_out = base == inner, base == outer
        assert np.all(is_in | is_out)
        if 0 < rank < nparts - 1:
            n_in, n_out = int(np.sum(is_in & ~is_out)), int(np.sum(is_out & ~is_in))
            assert n_in == n_out == R // 2          # half of the rows run inside-out (eq. 11), half outside-in (eq. 12)


def test_shard_argument_errors(E):
    import ctypes as C
    L = E.lib()
    R = E.etics_mex_shard_rows(3)
    assert R > 0 and E.etics_mex_shard_rows(-1) == 0 and E.etics_mex_shard_rows(E.ETICS_MAX_LMAX + 1) == 0
    parts = torch.zeros((2, R), dtype=torch.float64, device="cuda")
    base = torch.zeros(R, dtype=torch.float64, device="cuda")
    assert L.etics_mex_shard_bases(parts.data_ptr(), 2, 2, 3, base.data_ptr(), None) == E.ETICS_ERR_ARG      # rank out of range
    assert L.etics_mex_shard_bases(parts.data_ptr(), 0, 0, 3, base.data_ptr(), None) == E.ETICS_ERR_ARG
    assert L.etics_mex_shard_bases(parts.data_ptr(), 2, 0, 11, base.data_ptr(), None) == E.ETICS_ERR_LIMIT
    assert L.etics_mex_shard_bases(None, 2, 0, 3, base.data_ptr(), None) == E.ETICS_ERR_ARG
    ws = workspace(E, 100, 3)
    pos = torch.ones((3, 100), dtype=torch.float64, device="cuda")
    assert L.etics_mex_shard_moments(pos.data_ptr(), pos.data_ptr(), 100, 3, base.data_ptr(), ws.data_ptr(), 16, None) == E.ETICS_ERR_WORKSPACE
    assert L.etics_mex_shard_moments(pos.data_ptr(), pos.data_ptr(), 0, 3, base.data_ptr(), ws.data_ptr(), ws.numel(), None) == E.ETICS_ERR_ARG
    acc = torch.zeros((3, 100), dtype=torch.float64, device="cuda")
    assert L.etics_mex_shard_force(100, 3, 7, base.data_ptr(), acc.data_ptr(), acc.data_ptr(), ws.data_ptr(), ws.numel(), None) == E.ETICS_ERR_ARG
    assert L.etics_mex_shard_force(100, 3, 0, None, acc.data_ptr(), acc.data_ptr(), ws.data_ptr(), ws.numel(), None) == E.ETICS_ERR_ARG
    assert L.etics_mex_shard_force(100, 3, 0, base.data_ptr() + 8, acc.data_ptr(), acc.data_ptr(), ws.data_ptr(), ws.numel(), None) == E.ETICS_ERR_ALIGN


ONE_RANK_WORKER = r"""
import os, sys
sys.path.insert(0, os.environ["ETICS_ROOT"]); sys.path.insert(0, os.path.join(os.environ["ETICS_ROOT"], "tests"))
import numpy as np, torch, torch.distributed as dist
import oracle
from paper_1406_4254_b200 import sharded, workloads as W
from parity import TOL, rel_err_scalar, rel_err_vector
torch.cuda.set_device(0)
dist.init_process_group("nccl", init_method="tcp://127.0.0.1:" + sys.argv[1], rank=0, world_size=1)
pos, mass = W.particles("hernquist", 40003, seed=11)
acc, pot = sharded.mex_force_sharded(torch.from_numpy(pos).cuda(), torch.from_numpy(mass).cuda(), 6)
torch.cuda.synchronize()
acc0, pot0 = oracle.mex_force(pos, mass, 6)
ep, ea = rel_err_scalar(pot.cpu().numpy(), pot0, floor=0.0), rel_err_vector(acc.cpu().numpy(), acc0)
dist.destroy_process_group()
print("ERR", ep, ea, flush=True)
assert ep <= TOL and ea <= TOL
"""


def test_sharded_driver_with_the_real_kernels_one_rank(tmp_path):
    """paper_1406_4254_b200.sharded.mex_force_sharded end to end (sort, sample, all-to-all, moments, all-gather, bases, force,
    all-to-all back) over NCCL with a world of one rank — the one configuration a one-GPU box can run."""
    import socket
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        port = s.getsockname()[1]
    w = tmp_path / "one_rank.py"
    w.write_text(ONE_RANK_WORKER)
    r = subprocess.run([sys.executable, str(w), str(port)], capture_output=True, text=True, timeout=600,
                       env=dict(os.environ, ETICS_ROOT=ROOT), cwd=ROOT)
    assert r.returncode == 0, (r.stdout[-1000:], r.stderr[-3000:])
