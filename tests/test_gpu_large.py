"""GPU-vs-oracle parity at the FULL sizes of BASELINE.json configs[3] (N = 10^7, SCF (20,10), triaxial) and
configs[4] (N = 10^8 Plummer: SCF (10,6) and MEX lmax = 8), in the launch configuration bench.py times
(`--workload c4` / `--workload c5`), through the C ABI.

What the oracle can do at these sizes: the coefficient pass in full (OpenMP, seconds), the radial sort in full
(std::stable_sort), and potentials/accelerations of a SAMPLE of particles one by one — SCF evaluation is
per-particle independent; for MEX `oracle.mex_force_at` sums eqs. 11-12 over all N particles for each sampled
particle straight from the definition.  Samples: the extremes (innermost, outermost, closest to the z axis) plus a
strided set that spans tiles and the ragged tail.
"""
import numpy as np
import pytest

import oracle
from paper_1406_4254_b200 import workloads as W
from parity import TOL, rel_err_scalar, rel_err_vector

torch = pytest.importorskip("torch")
pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def E():
    assert torch.cuda.is_available(), "GPU tests need a CUDA device"
    from paper_1406_4254_b200 import binding
    binding.lib()
    binding.etics_init()
    return binding


def sample_indices(pos, stride, extremes=24):
    n = pos.shape[1]
    r2 = np.sum(pos ** 2, axis=0)
    sth2 = (pos[0] ** 2 + pos[1] ** 2) / r2
    return np.unique(np.concatenate([np.argpartition(r2, extremes)[:extremes], np.argpartition(-r2, extremes)[:extremes],
                                     np.argpartition(sth2, extremes)[:extremes], np.arange(0, n, stride),
                                     np.arange(n - 40, n)]))


def scf_full_size(E, pos, mass, nmax, lmax, stride):
    n = len(mass)
    dpos, dmass = torch.from_numpy(pos).cuda(), torch.from_numpy(mass).cuda()
    A, B = E.etics_scf_coeffs(dpos, dmass, nmax, lmax)
    acc, pot = E.etics_scf_force(dpos, nmax, lmax, A, B)
    torch.cuda.synchronize()
    A, B = A.cpu().numpy(), B.cpu().numpy()
    assert bool(torch.isfinite(acc).all()) and bool(torch.isfinite(pot).all())
    A0, B0 = oracle.scf_coeffs(pos, mass, nmax, lmax)
    assert rel_err_scalar(A, A0) <= TOL and rel_err_scalar(B, B0) <= TOL
    idx = sample_indices(pos, stride)
    acc0, pot0 = oracle.scf_force(np.ascontiguousarray(pos[:, idx]), nmax, lmax, A0, B0)
    didx = torch.from_numpy(idx).cuda()
    assert rel_err_scalar(pot[didx].cpu().numpy(), pot0, floor=0.0) <= TOL
    assert rel_err_vector(acc[:, didx].cpu().numpy(), acc0) <= TOL
    return A0


def test_config4_full_size_triaxial_nmax20_lmax10(E):
    """configs[3]: N = 10^7 triaxial Hernquist (1, 0.8, 0.6), (nmax, lmax) = (20, 10): T = 1386 coefficients, the
    multi-group accumulate path and the 44 KB evaluation table; even-l, even-m terms are O(1)."""
    c = W.CONFIGS[4]
    pos, mass = W.config_particles(4)
    A0 = scf_full_size(E, pos, mass, c["nmax"], c["lmax"], stride=9973)
    L = oracle.num_lm(c["lmax"])
    assert abs(A0[oracle.lm_index(2, 0)]) > 1e-3 and abs(A0[oracle.lm_index(2, 2)]) > 1e-4   # the triaxial signal is there
    assert abs(A0[oracle.lm_index(1, 0)]) < 1e-2 and L == 66


@pytest.fixture(scope="module")
def plummer_1e8():
    return W.config_particles(5)


def test_config5_scf_full_size(E, plummer_1e8):
    """configs[4], SCF half: N = 10^8 Plummer sphere, (10,6).  Also the Plummer closed form of pin P5:
    E[A_000] = 1.3047063, sigma = 0.5048/sqrt(N)."""
    pos, mass = plummer_1e8
    A0 = scf_full_size(E, pos, mass, 10, 6, stride=99_991)
    assert abs(A0[0] - 1.3047063) < 4 * 0.5048 / np.sqrt(len(mass)) + 1e-7


def test_config5_mex_full_size(E, plummer_1e8):
    """configs[4], MEX half: N = 10^8, lmax = 8.  Sort permutation and sorted keys bit-exact against the oracle's
    full std::stable_sort; potential and acceleration on sampled particles against the definition."""
    pos, mass = plummer_1e8
    n = len(mass)
    dpos, dmass = torch.from_numpy(pos).cuda(), torch.from_numpy(mass).cuda()
    keys, perm = E.etics_mex_sort(dpos)
    torch.cuda.synchronize()
    keys, perm = keys.cpu().numpy().view(np.uint64), perm.cpu().numpy().view(np.uint32)
    keys0, perm0 = oracle.mex_sort(pos)
    assert np.array_equal(perm, perm0), "sort permutation is not bit-exact at N = 10^8"
    assert np.array_equal(keys, keys0)
    del keys, perm, keys0
    acc, pot = E.etics_mex_force(dpos, dmass, 8)
    torch.cuda.synchronize()
    assert bool(torch.isfinite(acc).all()) and bool(torch.isfinite(pot).all())
    # samples: extremes in index space and in RANK space (first/last tiles of the sorted list), plus a strided set
    idx = np.unique(np.concatenate([sample_indices(pos, 4_999_999, extremes=6), perm0[:4].astype(np.int64),
                                    perm0[-4:].astype(np.int64), perm0[n // 2: n // 2 + 2].astype(np.int64)]))
    acc0, pot0 = oracle.mex_force_at(pos, mass, 8, idx)
    didx = torch.from_numpy(idx).cuda()
    assert rel_err_scalar(pot[didx].cpu().numpy(), pot0, floor=0.0) <= TOL
    assert rel_err_vector(acc[:, didx].cpu().numpy(), acc0) <= TOL


def test_config5_mex_in_four_radius_shards(E, plummer_1e8):
    """configs[4], MEX half, as the four ranks of a radius-partitioned run would see it: the
    N = 10^8 particles split into four radius ranges, every range through etics_mex_shard_moments / _bases / _force one after the
    other on this GPU, sampled particles of every range (its first and last ranks included) against the definition."""
    pos, mass = plummer_1e8
    n = len(mass)
    lmax = 8
    keys0, perm0 = oracle.mex_sort(pos)
    edges = [0]
    for c in (n // 4, n // 2 + 12_345, 3 * (n // 4)):
        while keys0[c] == keys0[c - 1]:      # equal keys stay in one shard
            c += 1
        edges.append(c)
    edges.append(n)
    R = E.etics_mex_shard_rows(lmax)
    parts = torch.zeros((4, R), dtype=torch.float64, device="cuda")
    shards, state = [], []
    for s in range(4):
        idx = np.sort(perm0[edges[s]:edges[s + 1]].astype(np.int64))     # a shard keeps the order of the particles' indices
        ws = torch.empty(E.etics_workspace_bytes(E.ETICS_WS_MEX_FORCE, len(idx), 0, lmax), dtype=torch.uint8, device="cuda")
        E.etics_mex_shard_moments(torch.from_numpy(np.ascontiguousarray(pos[:, idx])).cuda(), torch.from_numpy(mass[idx]).cuda(),
                                  lmax, ws, totals=parts[s])
        shards.append(idx)
        state.append(ws)
    torch.cuda.synchronize()
    got_idx, got_acc, got_pot = [], [], []
    for s in range(4):
        idx = shards[s]
        acc, pot = E.etics_mex_shard_force(len(idx), lmax, E.ETICS_WHAT_BOTH, E.etics_mex_shard_bases(parts, s, lmax), state[s])
        torch.cuda.synchronize()
        assert bool(torch.isfinite(acc).all()) and bool(torch.isfinite(pot).all())
        # samples of this range: its innermost and outermost particles and a few in between (global indices)
        ranks = np.unique(np.concatenate([np.arange(edges[s], edges[s] + 2), np.arange(edges[s + 1] - 2, edges[s + 1]),
                                          np.linspace(edges[s], edges[s + 1] - 1, 5).astype(np.int64)]))
        g = perm0[ranks].astype(np.int64)
        loc = torch.from_numpy(np.searchsorted(idx, g)).cuda()
        got_idx.append(g); got_acc.append(acc[:, loc].cpu().numpy()); got_pot.append(pot[loc].cpu().numpy())
        state[s] = None
    g = np.concatenate(got_idx)
    acc0, pot0 = oracle.mex_force_at(pos, mass, lmax, g)
    assert rel_err_scalar(np.concatenate(got_pot), pot0, floor=0.0) <= TOL
    assert rel_err_vector(np.concatenate(got_acc, axis=1), acc0) <= TOL
