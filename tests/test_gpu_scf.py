"""GPU-vs-oracle parity for the SCF half of the hot path, through the C ABI (binding -> libetics.so).

Same seeded inputs on both sides (paper_1406_4254_b200.workloads); tolerance = north_star's 1e-10 with the
metric of tests/parity.py (reading G13).  Expected values always come from oracle/, never from the CUDA path.
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
    binding.lib()          # fails loudly if libetics.so is missing: there is no fallback
    binding.etics_init()
    return binding


def dev(a):
    return torch.from_numpy(np.ascontiguousarray(a)).cuda()


def gpu_scf(E, pos, mass, nmax, lmax):
    dpos, dmass = dev(pos), dev(mass)
    A, B = E.etics_scf_coeffs(dpos, dmass, nmax, lmax)
    acc, pot = E.etics_scf_force(dpos, nmax, lmax, A, B)
    torch.cuda.synchronize()
    return A.cpu().numpy(), B.cpu().numpy(), acc.cpu().numpy(), pot.cpu().numpy()


def check_scf(E, pos, mass, nmax, lmax, tol=TOL):
    A, B, acc, pot = gpu_scf(E, pos, mass, nmax, lmax)
    A0, B0 = oracle.scf_coeffs(pos, mass, nmax, lmax)
    assert rel_err_scalar(A, A0) <= tol
    # B_{nl0} is written as +0.0 on both sides; the floor-scaled metric covers the rest
    L = oracle.num_lm(lmax)
    m0 = [n * L + oracle.lm_index(l, 0) for n in range(nmax + 1) for l in range(lmax + 1)]
    assert np.all(B[m0] == 0.0) and np.all(B0[m0] == 0.0)
    if lmax > 0:
        assert rel_err_scalar(B, B0) <= tol
    # evaluation from the GPU's own coefficients (full force calculation) ...
    acc0, pot0 = oracle.scf_force(pos, nmax, lmax, A0, B0)
    assert rel_err_scalar(pot, pot0, floor=0.0) <= tol
    assert rel_err_vector(acc, acc0) <= tol
    return A, B, acc, pot


def test_config1_hernquist_1e4(E):
    """BASELINE.json configs[0]: N=10^4 Hernquist, (nmax,lmax)=(10,6), seed 0."""
    pos, mass = W.config_particles(1)
    A, B, acc, pot = check_scf(E, pos, mass, 10, 6)
    # pin P5 on the GPU result too: A_000 = 3 E[1/(1+r)] = 303/301 within Monte-Carlo error
    assert abs(A[0] - 303.0 / 301.0) < 4 * 0.7048 / np.sqrt(len(mass))


def test_eval_alone_with_oracle_coefficients(E):
    """etics_scf_force on field points that are not the particles, coefficients from the oracle."""
    pos, mass = W.config_particles(1, n=5000)
    A0, B0 = oracle.scf_coeffs(pos, mass, 10, 6)
    pts, _ = W.particles("plummer", 3001, seed=7, axes=(1.0, 0.7, 1.3))
    acc, pot = E.etics_scf_force(dev(pts), 10, 6, dev(A0), dev(B0))
    acc0, pot0 = oracle.scf_force(pts, 10, 6, A0, B0)
    assert rel_err_scalar(pot.cpu().numpy(), pot0, floor=0.0) <= TOL
    assert rel_err_vector(acc.cpu().numpy(), acc0) <= TOL


@pytest.mark.parametrize("nmax,lmax", [(0, 0), (1, 0), (0, 1), (3, 2), (5, 2), (10, 6), (7, 9), (20, 10), (32, 10), (32, 3)])
def test_cutoffs(E, nmax, lmax):
    """Every lmax template instance and the n-chunking of the accumulate kernel; triaxial so that all even
    (l,m) terms are O(1) (config 4's shape)."""
    pos, mass = W.particles("hernquist", 4099, seed=3, axes=(1.0, 0.8, 0.6))
    check_scf(E, pos, mass, nmax, lmax)


@pytest.mark.parametrize("lmax", range(0, 11))
def test_every_lmax(E, lmax):
    pos, mass = W.particles("plummer", 1531, seed=11, axes=(0.9, 1.0, 0.5))
    check_scf(E, pos, mass, 4, lmax)


@pytest.mark.parametrize("lmax", range(0, 8))
def test_nmax10_every_lmax(E, lmax):
    """nmax = 10 selects the evaluation kernel with fully unrolled n loops for lmax <= 6 (monic Gegenbauer recurrence,
    scales folded into the coefficient table); lmax = 7 takes the run-time loop at the same nmax."""
    pos, mass = W.particles("hernquist", 2777, seed=13, axes=(1.0, 0.7, 0.9))
    check_scf(E, pos, mass, 10, lmax)


@pytest.mark.parametrize("n", [1, 2, 31, 32, 33, 63, 64, 65, 127, 129, 1000, 37889])
def test_ragged_sizes(E, n):
    """Sizes around the pass (32/64 particles) and block boundaries, including a single particle."""
    pos, mass = W.particles("hernquist", n, seed=5, axes=(1.0, 0.9, 0.7))
    mass = mass * (1.0 + 0.5 * np.sin(np.arange(n)))        # unequal masses
    check_scf(E, pos, mass, 6, 4)


def test_on_axis_and_extreme_particles(E):
    """On-axis particles (x=y=0 -> phi := 0, reading G10), near-axis (theta ~ 1e-7), tiny and huge radii."""
    pos = np.array([
        [0.0, 0.0, 1e-7, 1e-9, 0.3, 1e-5, 250.0, 0.0, -1e-8, 2e-4],
        [0.0, 0.0, 0.0, 1e-9, -0.4, 1e-5, 100.0, 1e-7, 1e-8, 1e-4],
        [1.0, -2.5, 1.0, 1.0, 0.5, 1e-5, -120.0, -3.0, 0.7, -1e-4],
    ])
    mass = np.linspace(0.05, 0.15, pos.shape[1])
    check_scf(E, pos, mass, 10, 10)
    check_scf(E, pos, mass, 10, 6)


def test_deterministic_bitwise(E):
    """No fp64 atomics: two calls on the same input give bit-identical A, B, acc, pot."""
    pos, mass = W.config_particles(1, n=50_000)
    r1 = gpu_scf(E, pos, mass, 10, 6)
    r2 = gpu_scf(E, pos, mass, 10, 6)
    for a, b in zip(r1, r2):
        assert np.array_equal(a, b)


def test_inputs_not_modified_and_caller_stream(E):
    pos, mass = W.config_particles(1, n=3000)
    dpos, dmass = dev(pos), dev(mass)
    st = torch.cuda.Stream()
    with torch.cuda.stream(st):
        A, B = E.etics_scf_coeffs(dpos, dmass, 10, 6, stream=st)
        acc, pot = E.etics_scf_force(dpos, 10, 6, A, B, stream=st)
    st.synchronize()
    assert np.array_equal(dpos.cpu().numpy(), pos) and np.array_equal(dmass.cpu().numpy(), mass)
    A0, B0 = oracle.scf_coeffs(pos, mass, 10, 6)
    assert rel_err_scalar(A.cpu().numpy(), A0) <= TOL


def test_host_entry_point(E):
    """etics_scf_full_host: HOST buffers in and out (the end-to-end path bench.py times as `e2e`)."""
    pos, mass = W.config_particles(1, n=20_000)
    n = len(mass)
    T = 11 * 28
    pos_h = torch.from_numpy(pos).pin_memory()
    mass_h = torch.from_numpy(mass).pin_memory()
    acc_h = torch.empty((3, n), dtype=torch.float64).pin_memory()
    pot_h = torch.empty(n, dtype=torch.float64).pin_memory()
    A_h = torch.empty(T, dtype=torch.float64).pin_memory()
    B_h = torch.empty(T, dtype=torch.float64).pin_memory()
    scratch = torch.empty(E.etics_host_scratch_bytes(0, n, 10, 6), dtype=torch.uint8, device="cuda")
    E.etics_scf_full_host(pos_h, mass_h, 10, 6, acc_h, pot_h, scratch, A_h, B_h)
    torch.cuda.synchronize()
    A0, B0 = oracle.scf_coeffs(pos, mass, 10, 6)
    acc0, pot0 = oracle.scf_force(pos, 10, 6, A0, B0)
    assert rel_err_scalar(A_h.numpy(), A0) <= TOL
    assert rel_err_scalar(pot_h.numpy(), pot0, floor=0.0) <= TOL
    assert rel_err_vector(acc_h.numpy(), acc0) <= TOL


def test_config2_full_size_sampled(E):
    """BASELINE.json configs[1] at full size (N=10^6), the launch configuration bench.py times.
    Coefficients against the full oracle pass (a few seconds, all cores); potential/acceleration on a
    sample of particles the oracle evaluates one by one (the evaluation is per-particle independent)."""
    pos, mass = W.config_particles(2)
    A, B, acc, pot = gpu_scf(E, pos, mass, 10, 6)
    A0, B0 = oracle.scf_coeffs(pos, mass, 10, 6)
    assert rel_err_scalar(A, A0) <= TOL and rel_err_scalar(B, B0) <= TOL
    n = len(mass)
    # sample: the extremes (smallest/largest r, closest to the z axis) plus a strided subset spanning tiles
    r = np.sqrt(np.sum(pos ** 2, axis=0))
    sth = np.sqrt(pos[0] ** 2 + pos[1] ** 2) / r
    idx = np.unique(np.concatenate([np.argsort(r)[:50], np.argsort(r)[-50:], np.argsort(sth)[:50],
                                    np.arange(0, n, 997), np.arange(n - 300, n)]))
    acc0, pot0 = oracle.scf_force(pos[:, idx], 10, 6, A0, B0)
    assert rel_err_scalar(pot[idx], pot0, floor=0.0) <= TOL
    assert rel_err_vector(acc[:, idx], acc0) <= TOL
    assert np.all(np.isfinite(acc)) and np.all(np.isfinite(pot))
    assert abs(A[0] - 303.0 / 301.0) < 4 * 0.7048 / np.sqrt(n)


@pytest.mark.parametrize("nmax,lmax", [(10, 6), (7, 3), (20, 10), (10, 8), (0, 0)])
def test_force_only_and_potential_only(E, nmax, lmax):
    """PAPER.md:253 ("force, potential or both"): the selector variants against the oracle, and bit-identical to the
    corresponding outputs of the 'both' call; the array that is not asked for is not touched."""
    pos, mass = W.particles("hernquist", 5_003, seed=7, axes=(1.0, 0.9, 0.7))
    dpos, dmass = dev(pos), dev(mass)
    A, B = E.etics_scf_coeffs(dpos, dmass, nmax, lmax)
    acc, pot = E.etics_scf_force(dpos, nmax, lmax, A, B)
    sentinel = -12345.0
    acc_p = torch.full_like(acc, sentinel)
    _, pot_p = E.etics_scf_force_ex(dpos, nmax, lmax, A, B, E.ETICS_WHAT_POTENTIAL, acc=None)
    pot_f = torch.full_like(pot, sentinel)
    acc_f, _ = E.etics_scf_force_ex(dpos, nmax, lmax, A, B, E.ETICS_WHAT_FORCE, pot=None)
    # arrays passed but not asked for stay untouched
    E.lib().etics_scf_force_ex(dpos.data_ptr(), pos.shape[1], nmax, lmax, A.data_ptr(), B.data_ptr(), E.ETICS_WHAT_POTENTIAL,
                               acc_p.data_ptr(), pot_p.data_ptr(), None, 0, torch.cuda.current_stream().cuda_stream)
    E.lib().etics_scf_force_ex(dpos.data_ptr(), pos.shape[1], nmax, lmax, A.data_ptr(), B.data_ptr(), E.ETICS_WHAT_FORCE,
                               acc_f.data_ptr(), pot_f.data_ptr(), None, 0, torch.cuda.current_stream().cuda_stream)
    torch.cuda.synchronize()
    assert torch.all(acc_p == sentinel) and torch.all(pot_f == sentinel)
    A0, B0 = oracle.scf_coeffs(pos, mass, nmax, lmax)
    acc0, pot0 = oracle.scf_force(pos, nmax, lmax, A0, B0)
    assert rel_err_scalar(pot_p.cpu().numpy(), pot0, floor=0.0) <= TOL
    assert rel_err_vector(acc_f.cpu().numpy(), acc0) <= TOL
    assert torch.equal(acc_f, acc)
    assert rel_err_scalar(pot_p.cpu().numpy(), pot.cpu().numpy(), floor=0.0) <= 1e-14   # same sums, possibly another schedule
    assert E.lib().etics_scf_force_ex(dpos.data_ptr(), pos.shape[1], nmax, lmax, A.data_ptr(), B.data_ptr(), 3,
                                      acc.data_ptr(), pot.data_ptr(), None, 0, 0) == E.ETICS_ERR_ARG


def test_sharded_scf_on_one_gpu_matches_the_whole(E):
    """etics_scf_combine + the shard arithmetic of paper_1406_4254_b200.sharded, with both 'ranks' on this GPU one after the
    other (no process group): shard tables added in rank order = coefficients of the whole set; shard evaluations = slices."""
    from paper_1406_4254_b200 import sharded
    n, nmax, lmax, world = 50_001, 10, 6, 3
    pos, mass = W.particles("hernquist", n, seed=9, axes=(1.0, 0.8, 0.6))
    T = (nmax + 1) * E.num_lm(lmax)
    tables = torch.empty((world, 2 * T), dtype=torch.float64, device="cuda")
    shards = []
    for r in range(world):
        a, b = sharded.shard_range(n, r, world)
        dp, dm = dev(pos[:, a:b]), dev(mass[a:b])
        E.etics_scf_coeffs(dp, dm, nmax, lmax, tables[r, :T], tables[r, T:])
        shards.append((a, b, dp))
    table = sharded.gather_and_combine(tables[0], lambda t: tables, E.etics_scf_combine)
    A0, B0 = oracle.scf_coeffs(pos, mass, nmax, lmax)
    assert rel_err_scalar(table[:T].cpu().numpy(), A0) <= TOL and rel_err_scalar(table[T:].cpu().numpy(), B0) <= TOL
    expect = tables[0].clone()
    for r in range(1, world):
        expect += tables[r]
    assert torch.equal(table, expect)                     # rank order, one addition per rank
    acc0, pot0 = oracle.scf_force(pos, nmax, lmax, A0, B0)
    for a, b, dp in shards:
        acc, pot = E.etics_scf_force(dp, nmax, lmax, table[:T].contiguous(), table[T:].contiguous())
        assert rel_err_vector(acc.cpu().numpy(), acc0[:, a:b]) <= TOL
        assert rel_err_scalar(pot.cpu().numpy(), pot0[a:b], floor=0.0) <= TOL


F32_TOL_POT, F32_TOL_ACC = 1e-4, 1e-3   # fp32 eps 6e-8 x the ~1e3 cancellation of the mixed-sign sums over (n, l, m); see DESIGN.md


@pytest.mark.parametrize("nmax,lmax", [(10, 6), (20, 10), (6, 2), (0, 0)])
def test_f32_mode_against_the_fp64_oracle(E, nmax, lmax):
    """single-precision evaluation; coefficients from the fp64 path."""
    pos, mass = W.particles("hernquist", 20_011, seed=17, axes=(1.0, 0.8, 0.6))
    dpos, dmass = dev(pos), dev(mass)
    A, B = E.etics_scf_coeffs(dpos, dmass, nmax, lmax)
    acc, pot = E.etics_scf_force_f32(dpos, nmax, lmax, A, B)
    _, pot_only = E.etics_scf_force_f32(dpos, nmax, lmax, A, B, E.ETICS_WHAT_POTENTIAL)
    acc_only, _ = E.etics_scf_force_f32(dpos, nmax, lmax, A, B, E.ETICS_WHAT_FORCE)
    torch.cuda.synchronize()
    A0, B0 = oracle.scf_coeffs(pos, mass, nmax, lmax)
    acc0, pot0 = oracle.scf_force(pos, nmax, lmax, A0, B0)
    ep, ea = rel_err_scalar(pot.cpu().numpy(), pot0, floor=0.0), rel_err_vector(acc.cpu().numpy(), acc0)
    assert ep <= F32_TOL_POT and ea <= F32_TOL_ACC, (ep, ea)
    assert ep > 1e-9          # it really is single precision
    assert torch.equal(pot_only, pot) and torch.equal(acc_only, acc)


def test_f32_mode_is_accurate_near_the_z_axis(E):
    """the paper's fp32 runs fail near the z axis (eq. 24); the l-recurrence at fixed m does not."""
    nmax, lmax = 10, 6
    pos, mass = W.config_particles(1)
    A, B = E.etics_scf_coeffs(dev(pos), dev(mass), nmax, lmax)
    # field points: on the axis, and 1e-7 ... 1e-2 rad off it, both poles, several radii
    th = np.array([0.0, 1e-7, 1e-5, 1e-4, 1e-3, 1e-2])
    th = np.concatenate([th, np.pi - th])
    r = np.array([0.05, 0.7, 3.0, 40.0])
    T, R = np.meshgrid(th, r, indexing="ij")
    ph = 0.3 + 1.7 * np.arange(T.size)
    pts = np.stack([(R * np.sin(T)).ravel() * np.cos(ph), (R * np.sin(T)).ravel() * np.sin(ph), (R * np.cos(T)).ravel()])
    acc, pot = E.etics_scf_force_f32(dev(pts), nmax, lmax, A, B)
    torch.cuda.synchronize()
    A0, B0 = oracle.scf_coeffs(pos, mass, nmax, lmax)
    acc0, pot0 = oracle.scf_force(pts, nmax, lmax, A0, B0)
    assert rel_err_scalar(pot.cpu().numpy(), pot0, floor=0.0) <= F32_TOL_POT
    assert rel_err_vector(acc.cpu().numpy(), acc0) <= F32_TOL_ACC
