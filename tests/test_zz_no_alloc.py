"""etics_scf_coeffs_static: the SCF coefficients without a caller workspace (block partials in the library's own
__device__ array; include/etics.h).  Collected LAST on purpose (the file name): a failure here must not hide other tests
under `pytest -x`.

Compared against the existing path (etics_scf_coeffs with a caller workspace: the same kernels, so the tables must be
bit-identical, which is inside the 1e-10 of every other parity test) and against the oracle, on two calls in a row
with DIFFERENT sizes, after a call that leaves NaN in every partial of the shared array: a result that depended on
the array's previous contents would fail.
"""
import numpy as np
import pytest

import oracle
from paper_1406_4254_b200 import workloads as W
from parity import TOL, rel_err_scalar

torch = pytest.importorskip("torch")
pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def E():
    assert torch.cuda.is_available(), "GPU tests need a CUDA device"
    from paper_1406_4254_b200 import binding
    binding.lib()          # fails loudly if libetics.so is missing: there is no fallback
    return binding         # no etics_init(): the entry point must do its own per-device set-up when run alone


def dev(a):
    return torch.from_numpy(np.ascontiguousarray(a)).cuda()


def static_coeffs(E, dpos, dmass, nmax, lmax):
    T = (nmax + 1) * E.num_lm(lmax)
    A = torch.full((T,), float("nan"), dtype=torch.float64, device="cuda")
    B = torch.full((T,), float("nan"), dtype=torch.float64, device="cuda")
    E.etics_scf_coeffs_static(dpos, dmass, nmax, lmax, A, B)
    return A, B


def test_static_scratch_matches_workspace_path_two_calls_in_a_row(E):
    cases = [(20000, 20, 10, 3), (777, 10, 6, 4), (20000, 20, 10, 5)]   # largest table allowed, a small one, the largest again
    # poison: NaN positions put NaN into every block partial of the shared array at the largest table
    N0 = 148 * 128 * 2
    poison = torch.full((3, N0), float("nan"), dtype=torch.float64, device="cuda")
    A, B = static_coeffs(E, poison, torch.ones(N0, dtype=torch.float64, device="cuda"), 20, 10)
    torch.cuda.synchronize()
    assert torch.isnan(A).all()
    for N, nmax, lmax, seed in cases:
        pos, mass = W.particles("hernquist", N, seed=seed)
        dpos, dmass = dev(pos), dev(mass)
        A, B = static_coeffs(E, dpos, dmass, nmax, lmax)
        A2, B2 = static_coeffs(E, dpos, dmass, nmax, lmax)       # second call in a row on the same array
        Aw, Bw = E.etics_scf_coeffs(dpos, dmass, nmax, lmax)    # the existing path: caller-allocated workspace
        torch.cuda.synchronize()
        A, B, A2, B2, Aw, Bw = (t.cpu().numpy() for t in (A, B, A2, B2, Aw, Bw))
        assert np.isfinite(A).all() and np.isfinite(B).all()
        assert np.array_equal(A, Aw) and np.array_equal(B, Bw)
        assert np.array_equal(A2, Aw) and np.array_equal(B2, Bw)
        A0, B0 = oracle.scf_coeffs(pos, mass, nmax, lmax)
        assert rel_err_scalar(A, A0) <= TOL
        assert rel_err_scalar(B, B0) <= TOL


def test_static_scratch_rejects_sizes_beyond_its_maximum(E):
    assert E.etics_scf_coeffs_static_max_table() == E.ETICS_STATIC_MAX_TABLE == 21 * 66
    pos, mass = W.particles("hernquist", 1000, seed=1)
    dpos, dmass = dev(pos), dev(mass)
    for nmax, lmax in [(21, 10), (32, 10), (32, 9)]:
        T = (nmax + 1) * E.num_lm(lmax)
        assert T > E.ETICS_STATIC_MAX_TABLE
        A = torch.full((T,), 7.0, dtype=torch.float64, device="cuda")
        B = torch.full((T,), 7.0, dtype=torch.float64, device="cuda")
        with pytest.raises(E.EticsError) as ei:
            E.etics_scf_coeffs_static(dpos, dmass, nmax, lmax, A, B)
        assert ei.value.status == E.ETICS_ERR_STATIC_LIMIT
        assert "ETICS_STATIC_MAX_TABLE" in str(ei.value)
        torch.cuda.synchronize()
        assert (A == 7.0).all() and (B == 7.0).all()   # nothing was launched
    # the largest sizes inside the limit are accepted: (20,10) above; (32,8) has T = 33 * 45 = 1485 > 1386, (29,8) = 1350
    A, B = static_coeffs(E, dpos, dmass, 29, 8)
    Aw, Bw = E.etics_scf_coeffs(dpos, dmass, 29, 8)
    torch.cuda.synchronize()
    assert torch.equal(A, Aw) and torch.equal(B, Bw)
