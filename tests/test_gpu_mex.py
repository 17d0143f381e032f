"""GPU-vs-oracle parity for the MEX half of the hot path, through the C ABI (binding -> libetics.so).

The sort permutation must be bit-exact (ties in r^2 broken by particle index, north_star); potentials and
accelerations within 1e-10 (tests/parity.py, reading G13).  Expected values come from oracle/ only.
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


def dev(a):
    return torch.from_numpy(np.ascontiguousarray(a)).cuda()


def gpu_sort(E, pos):
    keys, perm = E.etics_mex_sort(dev(pos))
    torch.cuda.synchronize()
    return keys.cpu().numpy().view(np.uint64), perm.cpu().numpy().view(np.uint32)


def check_sort(E, pos):
    keys, perm = gpu_sort(E, pos)
    keys0, perm0 = oracle.mex_sort(pos)
    assert np.array_equal(perm, perm0), "sort permutation is not bit-exact"
    assert np.array_equal(keys, keys0), "sorted keys differ"


def check_mex(E, pos, mass, lmax, tol=TOL):
    acc, pot = E.etics_mex_force(dev(pos), dev(mass), lmax)
    torch.cuda.synchronize()
    acc, pot = acc.cpu().numpy(), pot.cpu().numpy()
    acc0, pot0 = oracle.mex_force(pos, mass, lmax)
    n = len(mass)
    if n > 1:
        assert rel_err_scalar(pot, pot0, floor=0.0) <= tol
        assert rel_err_vector(acc, acc0) <= tol
    else:   # a single particle feels nothing (no self-interaction)
        assert np.all(pot == 0.0) and np.all(acc == 0.0) and np.all(pot0 == 0.0)
    return acc, pot


# ---------------------------------------------------------------------------------------------- sort
@pytest.mark.parametrize("n", [1, 2, 31, 255, 256, 257, 4095, 4096, 4097, 8191, 12289, 100_003])
def test_sort_sizes(E, n):
    """Sizes around the sort tile (4096 keys) and warp boundaries."""
    pos, _ = W.particles("hernquist", n, seed=2)
    check_sort(E, pos)


def test_sort_ties_broken_by_index(E):
    """Deliberate duplicate radii: mirrored pairs (+-z, permuted axes share r^2 bit for bit) and exact copies."""
    base, _ = W.particles("plummer", 5000, seed=4)
    pos = np.concatenate([base, -base, base[[1, 0, 2]], base * np.array([[1.0], [-1.0], [1.0]]), base], axis=1)
    rng = np.random.default_rng(0)
    pos = np.ascontiguousarray(pos[:, rng.permutation(pos.shape[1])])
    keys0, _ = oracle.mex_sort(pos)
    assert np.sum(keys0[1:] == keys0[:-1]) > 5000      # the input really has many exact ties
    check_sort(E, pos)


def test_sort_all_equal_and_extreme_keys(E):
    """All radii equal (one bucket in every pass: pure stability), and keys spanning the whole exponent range."""
    n = 9000
    pos = np.zeros((3, n)); pos[2] = 1.5
    check_sort(E, pos)
    expo = np.linspace(-150, 150, n)
    pos = np.zeros((3, n)); pos[0] = 10.0 ** expo[::-1]
    check_sort(E, pos)
    pos[0, ::7] = 0.0; pos[1, ::7] = 1e-170                  # r^2 underflows to 0: all such keys tie at 0
    check_sort(E, pos)


def _wide_range_with_clusters(sizes, jitter, seed):
    """Particles on the x axis: isolated ones spanning 40 octaves of r^2 (so that the sort drops the low key bits) plus
    clusters whose members differ only in those low bits (relative spacing `jitter`)."""
    rng = np.random.default_rng(seed)
    x = [10.0 ** rng.uniform(-3.0, 3.0, 4000)]
    for n in sizes:
        x0 = 10.0 ** rng.uniform(-2.0, 2.0)
        x.append(x0 * (1.0 + jitter * rng.permutation(n)))
    x = np.concatenate(x)
    pos = np.zeros((3, len(x)))
    pos[0] = x[rng.permutation(len(x))]
    return pos


def test_sort_prefix_collisions_short_runs(E):
    """Runs of 2..32 particles whose keys agree in the 33 sorted bits and differ below: the fix-up orders them."""
    rng = np.random.default_rng(5)
    pos = _wide_range_with_clusters(rng.integers(2, 33, 1500), 3e-13, seed=6)
    keys0, _ = oracle.mex_sort(pos)
    assert np.sum((keys0[1:] >> np.uint64(30)) == (keys0[:-1] >> np.uint64(30))) > 10_000   # many colliding neighbours
    check_sort(E, pos)


def test_sort_prefix_collisions_long_runs_fallback(E):
    """Runs longer than the fix-up handles (two thin shells of thousands of particles, and 100 exact copies of one
    particle) take the fallback sort; the result is the same bit-exact permutation."""
    pos = _wide_range_with_clusters([5000, 3000, 33], 1e-14, seed=7)
    check_sort(E, pos)
    pos = _wide_range_with_clusters([2], 1e-14, seed=8)
    pos = np.ascontiguousarray(np.concatenate([pos, np.repeat(pos[:, 17:18], 100, axis=1)], axis=1))
    check_sort(E, pos)


def _pad_to_bandwidth_bound_path(pos, n_total, seed):
    """The same clusters inside a set large enough (> ~1.2e6) for the one-kernel-per-phase sort (36 prefix bits, 9-bit digits)."""
    filler, _ = W.particles("hernquist", n_total - pos.shape[1], seed=seed)
    rng = np.random.default_rng(seed)
    allp = np.concatenate([pos, filler], axis=1)
    return np.ascontiguousarray(allp[:, rng.permutation(allp.shape[1])])


def test_sort_large_path_collisions_and_fallback(E):
    """The sort for N above one tile per resident block: short runs for the two-phase fix-up, exact duplicates, all-equal
    keys, and runs too long for the fix-up (fallback sort)."""
    rng = np.random.default_rng(15)
    pos = _pad_to_bandwidth_bound_path(_wide_range_with_clusters(rng.integers(2, 33, 3000), 2e-14, seed=16), 1_400_000, 17)
    keys0, _ = oracle.mex_sort(pos)
    assert np.sum((keys0[1:] >> np.uint64(27)) == (keys0[:-1] >> np.uint64(27))) > 20_000
    check_sort(E, pos)
    pos[:, 1000:1200] = pos[:, 999:1000]                     # 201 exact copies: a run the fix-up cannot order -> fallback
    check_sort(E, pos)
    pos = _pad_to_bandwidth_bound_path(_wide_range_with_clusters([4000, 64], 1e-15, seed=18), 1_300_001, 19)
    check_sort(E, pos)
    pos = np.zeros((3, 1_250_000)); pos[1] = 0.75             # every key equal: zero passes, pure stability
    check_sort(E, pos)


@pytest.mark.parametrize("n", [1_279_999, 1_280_000, 1_280_001, 1_515_520 + 4097])
def test_sort_large_path_tile_boundaries(E, n):
    """One-kernel-per-phase sort at sizes one below, at and one above a whole number of its 5120-word scatter tiles (250 of
    them), and one where the last segment holds a single ragged tile."""
    pos, _ = W.particles("hernquist", n, seed=23)
    check_sort(E, pos)


def test_sort_narrow_range_is_exact_without_fixup(E):
    """A thin shell: the whole key range fits the sorted prefix (shift = 0), whatever N."""
    rng = np.random.default_rng(11)
    v = rng.normal(size=(3, 30_000))
    pos = np.ascontiguousarray(v / np.sqrt(np.sum(v ** 2, axis=0)) * 1.25)
    check_sort(E, pos)


def test_sort_already_sorted_and_reversed(E):
    pos, _ = W.particles("hernquist", 20_000, seed=9)
    order = np.argsort(np.sum(pos ** 2, axis=0), kind="stable")
    check_sort(E, np.ascontiguousarray(pos[:, order]))
    check_sort(E, np.ascontiguousarray(pos[:, order[::-1]]))


def test_sort_config3_full_size(E):
    """BASELINE.json configs[2] input at full size: N = 10^6, bit-exact permutation."""
    pos, _ = W.config_particles(3)
    check_sort(E, pos)


# ---------------------------------------------------------------------------------------------- force
@pytest.mark.parametrize("lmax", range(0, 11))
def test_every_lmax(E, lmax):
    """Every lmax template instance / column grouping; triaxial so that all even (l,m) are O(1)."""
    pos, mass = W.particles("hernquist", 3001, seed=3, axes=(1.0, 0.8, 0.6))
    check_mex(E, pos, mass, lmax)


@pytest.mark.parametrize("n", [1, 2, 3, 7, 8, 9, 127, 1023, 1024, 1025, 2049, 10_000, 33_333])
def test_ragged_sizes(E, n):
    """Sizes around the chunk (8) and scan tile (1024) boundaries, including N = 1."""
    pos, mass = W.particles("plummer", n, seed=6, axes=(1.0, 0.9, 0.7))
    mass = mass * (1.0 + 0.5 * np.cos(np.arange(n)))        # unequal masses
    check_mex(E, pos, mass, 6)


def test_config3_shape_small(E):
    """configs[2]'s distribution and lmax at a size the oracle finishes in a second (several tiles + ragged tail)."""
    pos, mass = W.config_particles(3, n=50_001)
    check_mex(E, pos, mass, 6)


def test_lmax8_plummer(E):
    """configs[4]'s MEX leg (Plummer, lmax = 8) at reduced N."""
    pos, mass = W.config_particles(5, n=20_011)
    check_mex(E, pos, mass, 8)


def test_ties_and_on_axis(E):
    """Equal radii (exclusive sums must follow the index tie-break), on-axis and near-axis particles."""
    base, mass = W.particles("hernquist", 700, seed=12, axes=(1.0, 0.8, 0.6))
    pos = np.concatenate([base, -base, base * np.array([[1.0], [1.0], [-1.0]])], axis=1)
    extra = np.array([[0.0, 0.0, 1e-7, 0.0], [0.0, 0.0, 0.0, 1e-9], [0.5, -0.5, 2.0, 3.0]])
    pos = np.ascontiguousarray(np.concatenate([pos, extra], axis=1))
    mass = np.full(pos.shape[1], 1.0 / pos.shape[1])
    check_mex(E, pos, mass, 6)
    check_mex(E, pos, mass, 10)


def test_spherical_shells_lmax0(E):
    """Pin P10 on the GPU result itself: lmax = 0 is Gauss's law, a_r = -M(<r)/r^2."""
    pos, mass = W.particles("hernquist", 5000, seed=1)
    acc, pot = check_mex(E, pos, mass, 0)
    r = np.sqrt(np.sum(pos ** 2, axis=0))
    order = np.argsort(r, kind="stable")
    m_in = np.zeros_like(r); m_in[order] = np.concatenate([[0.0], np.cumsum(mass[order])[:-1]])
    a_r = np.sum(acc * pos, axis=0) / r
    assert np.allclose(a_r, -m_in / r ** 2, rtol=1e-12, atol=1e-300)


def test_deterministic_bitwise(E):
    pos, mass = W.config_particles(3, n=70_000)
    dp, dm = dev(pos), dev(mass)
    a1, p1 = E.etics_mex_force(dp, dm, 6)
    a2, p2 = E.etics_mex_force(dp, dm, 6)
    torch.cuda.synchronize()
    assert torch.equal(a1, a2) and torch.equal(p1, p2)
    assert np.array_equal(dp.cpu().numpy(), pos) and np.array_equal(dm.cpu().numpy(), mass)   # inputs untouched


def test_host_entry_point(E):
    pos, mass = W.config_particles(3, n=30_000)
    n = len(mass)
    pos_h = torch.from_numpy(pos).pin_memory()
    mass_h = torch.from_numpy(mass).pin_memory()
    acc_h = torch.empty((3, n), dtype=torch.float64).pin_memory()
    pot_h = torch.empty(n, dtype=torch.float64).pin_memory()
    scratch = torch.empty(E.etics_host_scratch_bytes(1, n, 0, 6), dtype=torch.uint8, device="cuda")
    E.etics_mex_full_host(pos_h, mass_h, 6, acc_h, pot_h, scratch)
    torch.cuda.synchronize()
    acc0, pot0 = oracle.mex_force(pos, mass, 6)
    assert rel_err_scalar(pot_h.numpy(), pot0, floor=0.0) <= TOL
    assert rel_err_vector(acc_h.numpy(), acc0) <= TOL


def test_config3_full_size(E):
    """BASELINE.json configs[2] at full size (N = 10^6, lmax = 6), the launch configuration bench.py times;
    the streaming oracle covers every particle in a few seconds."""
    pos, mass = W.config_particles(3)
    check_mex(E, pos, mass, 6)


@pytest.mark.parametrize("lmax", [0, 3, 6, 8, 10])
def test_force_only_and_potential_only(E, lmax):
    """PAPER.md:213 ("force, potential or both"): the selector variants against the oracle and against the 'both' call."""
    pos, mass = W.particles("hernquist", 4_321, seed=5, axes=(1.0, 0.8, 0.6))
    dpos, dmass = dev(pos), dev(mass)
    acc, pot = E.etics_mex_force(dpos, dmass, lmax)
    sentinel = -12345.0
    acc_p = torch.full_like(acc, sentinel)
    pot_f = torch.full_like(pot, sentinel)
    _, pot_p = E.etics_mex_force_ex(dpos, dmass, lmax, E.ETICS_WHAT_POTENTIAL)
    acc_f, _ = E.etics_mex_force_ex(dpos, dmass, lmax, E.ETICS_WHAT_FORCE)
    ws = torch.empty(E.etics_workspace_bytes(E.ETICS_WS_MEX_FORCE, pos.shape[1], 0, lmax), dtype=torch.uint8, device="cuda")
    st = torch.cuda.current_stream().cuda_stream
    assert E.lib().etics_mex_force_ex(dpos.data_ptr(), dmass.data_ptr(), pos.shape[1], lmax, E.ETICS_WHAT_POTENTIAL,
                                      acc_p.data_ptr(), pot_p.data_ptr(), ws.data_ptr(), ws.numel(), st) == 0
    assert E.lib().etics_mex_force_ex(dpos.data_ptr(), dmass.data_ptr(), pos.shape[1], lmax, E.ETICS_WHAT_FORCE,
                                      acc_f.data_ptr(), pot_f.data_ptr(), ws.data_ptr(), ws.numel(), st) == 0
    torch.cuda.synchronize()
    assert torch.all(acc_p == sentinel) and torch.all(pot_f == sentinel)
    acc0, pot0 = oracle.mex_force(pos, mass, lmax)
    assert rel_err_scalar(pot_p.cpu().numpy(), pot0, floor=0.0) <= TOL
    if lmax > 0:
        assert rel_err_vector(acc_f.cpu().numpy(), acc0) <= TOL
    assert torch.equal(acc_f, acc)
    assert rel_err_scalar(pot_p.cpu().numpy(), pot.cpu().numpy(), floor=0.0) <= 1e-14
    assert E.lib().etics_mex_force_ex(dpos.data_ptr(), dmass.data_ptr(), pos.shape[1], lmax, 7,
                                      acc.data_ptr(), pot.data_ptr(), ws.data_ptr(), ws.numel(), st) == E.ETICS_ERR_ARG


@pytest.mark.parametrize("two_streams", [False, True])
@pytest.mark.parametrize("n", [30_000, 400_003])
def test_step_host_entry_point(E, n, two_streams):
    """etics_step_host: one upload, both methods, overlapped copies — against the oracle, and bit-identical to the
    device-pointer calls (the upload is accumulated in ranges of whole blocks, so every block partial is unchanged)."""
    pos, mass = W.particles("hernquist", n, seed=3, axes=(1.0, 0.9, 0.8))
    pos_h, mass_h = torch.from_numpy(pos).pin_memory(), torch.from_numpy(mass).pin_memory()
    out = [torch.empty((3, n), dtype=torch.float64).pin_memory(), torch.empty(n, dtype=torch.float64).pin_memory(),
           torch.empty((3, n), dtype=torch.float64).pin_memory(), torch.empty(n, dtype=torch.float64).pin_memory()]
    T = 11 * E.num_lm(6)
    A_h, B_h = torch.empty(T, dtype=torch.float64).pin_memory(), torch.empty(T, dtype=torch.float64).pin_memory()
    scratch = torch.empty(E.etics_step_host_scratch_bytes(n, 10, 6, 4), dtype=torch.uint8, device="cuda")
    cs = torch.cuda.Stream() if two_streams else None
    for _ in range(2):   # a second call reuses the scratch while nothing is in flight
        E.etics_step_host(pos_h, mass_h, 10, 6, 4, out[0], out[1], out[2], out[3], scratch, A_h, B_h, copy_stream=cs)
        torch.cuda.current_stream().synchronize()
    dpos, dmass = dev(pos), dev(mass)
    A, B = E.etics_scf_coeffs(dpos, dmass, 10, 6)
    acc1, pot1 = E.etics_scf_force(dpos, 10, 6, A, B)
    acc2, pot2 = E.etics_mex_force(dpos, dmass, 4)
    torch.cuda.synchronize()
    for h, d in zip([A_h, B_h] + out, [A, B, acc1, pot1, acc2, pot2]):
        assert np.array_equal(h.numpy(), d.cpu().numpy())
    if n <= 30_000:
        A0, B0 = oracle.scf_coeffs(pos, mass, 10, 6)
        acc0, pot0 = oracle.scf_force(pos, 10, 6, A0, B0)
        assert rel_err_scalar(A_h.numpy(), A0) <= TOL and rel_err_vector(out[0].numpy(), acc0) <= TOL
        assert rel_err_scalar(out[1].numpy(), pot0, floor=0.0) <= TOL
        accm, potm = oracle.mex_force(pos, mass, 4)
        assert rel_err_vector(out[2].numpy(), accm) <= TOL and rel_err_scalar(out[3].numpy(), potm, floor=0.0) <= TOL
