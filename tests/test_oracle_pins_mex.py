"""Pins P10-P14 for the MEX half of the oracle: Gauss's law for shells, the pairwise
truncated Legendre series (exact at every lmax), convergence to brute-force Newtonian sums, the sort
against exact rational arithmetic, and the MEX<->SCF relation eq. (19).  CPU only."""
import math
from fractions import Fraction

import numpy as np
import pytest
from scipy import special

import oracle
from paper_1406_4254_b200 import workloads as W


def _direct_sum(pos, mass):
    """eq. (4) PAPER.md:82 and its gradient, no self-interaction."""
    d = pos[:, :, None] - pos[:, None, :]                  # x_i - x_j
    r2 = (d ** 2).sum(0)
    np.fill_diagonal(r2, np.inf)
    inv = 1.0 / np.sqrt(r2)
    pot = -(mass[None, :] * inv).sum(1)
    acc = -(mass[None, None, :] * d * inv[None] ** 3).sum(2)
    return acc, pot


def _pairwise_series_potential(xi, i, pos, mass, rank, lmax):
    """-sum_{j != i} m_j sum_{l<=lmax} r_<^l / r_>^(l+1) P_l(cos gamma) with the interior/exterior
    classification frozen by sorted rank (not by |xi|), evaluated at field point xi (long double)."""
    xi = np.asarray(xi, dtype=np.longdouble)
    r = np.sqrt((xi ** 2).sum())
    tot = np.longdouble(0)
    for j in range(pos.shape[1]):
        if j == i:
            continue
        pj = pos[:, j].astype(np.longdouble)
        rj = np.sqrt((pj ** 2).sum())
        cg = float((xi * pj).sum() / (r * rj))
        cg = max(-1.0, min(1.0, cg))
        # long-double Legendre P_l by Bonnet recurrence on the long-double cosine
        cgl = (xi * pj).sum() / (r * rj)
        pl_prev, pl = np.longdouble(1), cgl
        series = np.longdouble(0)
        for l in range(lmax + 1):
            if l == 0:
                p = np.longdouble(1)
            elif l == 1:
                p = cgl
            else:
                p = ((2 * l - 1) * cgl * pl - (l - 1) * pl_prev) / l
                pl_prev, pl = pl, p
            if rank[j] < rank[i]:
                series += p * rj ** l / r ** (l + 1)
            else:
                series += p * r ** l / rj ** (l + 1)
        tot -= np.longdouble(mass[j]) * series
    return tot


def test_P13_sort_keys_and_permutation_exact():
    # key = bits of fl(fl(fl(x*x) + y*y exact) + z*z exact): emulate with exact rationals + correct rounding
    pos, _ = W.particles("hernquist", 300, seed=2)
    # deliberate exact ties: mirrored pairs and +-z copies (same r^2 bit pattern), interleaved
    pos[:, 100:150] = -pos[:, 0:50]
    pos[:, 150:200] = pos[:, 50:100] * np.array([[1.0], [1.0], [-1.0]])
    pos[:, 200:220] = pos[:, 0:20]
    keys, perm = oracle.mex_sort(pos)
    exp_keys = np.empty(300, dtype=np.uint64)
    for k in range(300):
        x, y, z = (Fraction(float(v)) for v in pos[:, k])
        t = float(x * x)                       # float(Fraction) rounds to nearest-even
        t = float(y * y + Fraction(t))
        t = float(z * z + Fraction(t))
        exp_keys[k] = np.array([t]).view(np.uint64)[0]
    exp_perm = np.argsort(exp_keys, kind="stable").astype(np.uint32)
    assert np.array_equal(perm, exp_perm)
    assert np.array_equal(keys, exp_keys[exp_perm])
    # ties broken by original index (north_star): equal keys appear in increasing index order
    same = keys[1:] == keys[:-1]
    assert same.sum() >= 120
    assert np.all(perm[1:][same] > perm[:-1][same])
    assert sorted(perm.tolist()) == list(range(300))


def test_P10_monopole_is_gauss_law_for_shells():
    # lmax=0: a_r = -M(<r_i)/r_i^2, Phi_i = -M(<r_i)/r_i - sum_{j>i} m_j/r_j; strict inequalities (eqs. 11-12)
    rng = np.random.default_rng(5)
    n = 200
    pos = rng.normal(size=(3, n)) * rng.uniform(0.1, 3.0, size=n)
    mass = rng.uniform(0.5, 1.5, size=n)
    acc, pot = oracle.mex_force(pos, mass, 0)
    r = np.sqrt((pos ** 2).sum(0))
    order = np.argsort(r, kind="stable")
    rs, ms = r[order], mass[order]
    inner = np.concatenate([[0.0], np.cumsum(ms)[:-1]])
    outer = np.concatenate([np.cumsum((ms / rs)[::-1])[::-1][1:], [0.0]])
    exp_pot = np.empty(n); exp_ar = np.empty(n)
    exp_pot[order] = -inner / rs - outer
    exp_ar[order] = -inner / rs ** 2
    assert np.allclose(pot, exp_pot, rtol=1e-13)
    assert np.allclose(acc, exp_ar[None, :] * pos / r, rtol=1e-13, atol=1e-15)


@pytest.mark.parametrize("lmax", [0, 1, 2, 5, 8])
def test_P11_pairwise_truncated_series(lmax):
    # The (l,m) sums with w_lm collapse (addition theorem) to the pairwise Legendre series, exactly at every lmax.
    rng = np.random.default_rng(21)
    n = 40
    pos = rng.normal(size=(3, n)) * rng.uniform(0.2, 2.0, size=n)
    pos[:, 3] = [0.0, 0.0, 0.7]                 # on-axis particle
    pos[:, 4] = [1e-4, -2e-4, -1.1]             # near-axis particle
    pos[:, 6] = -pos[:, 5]                      # an exact tie in r^2: 5 counts as interior to 6
    mass = rng.uniform(0.5, 1.5, size=n) / n
    acc, pot, perm = oracle.mex_force(pos, mass, lmax, return_perm=True)
    rank = np.empty(n, dtype=np.int64); rank[perm] = np.arange(n)
    assert rank[5] < rank[6]
    for i in range(n):
        ref = _pairwise_series_potential(pos[:, i], i, pos, mass, rank, lmax)
        assert pot[i] == pytest.approx(float(ref), rel=1e-12, abs=1e-14)
    # acceleration = -gradient of that frozen-ordering function (long-double central differences)
    for i in (0, 3, 4, 5, 6, 17, 39):
        h = np.longdouble(1e-6) * np.sqrt((pos[:, i] ** 2).sum())
        g = np.zeros(3)
        for d in range(3):
            e = np.zeros(3, dtype=np.longdouble); e[d] = h
            xi = pos[:, i].astype(np.longdouble)
            fp = _pairwise_series_potential(xi + e, i, pos, mass, rank, lmax)
            fm = _pairwise_series_potential(xi - e, i, pos, mass, rank, lmax)
            fp2 = _pairwise_series_potential(xi + 2 * e, i, pos, mass, rank, lmax)
            fm2 = _pairwise_series_potential(xi - 2 * e, i, pos, mass, rank, lmax)
            g[d] = float((8 * (fp - fm) - (fp2 - fm2)) / (12 * h))
        assert np.allclose(acc[:, i], -g, rtol=1e-8, atol=1e-9 * np.abs(acc).max())


def test_P12_converges_to_newtonian_direct_sum():
    # well-separated radii r_k = 2^k/4 (1 + jitter): truncation error falls like (r_</r_>)^(lmax+1)  (north_star).
    # (fp64 holds the unnormalised P_lm ~ (2m-1)!! r^l up to lmax ~ 50 for this radius range.)
    rng = np.random.default_rng(9)
    n = 16
    rad = 0.25 * 2.0 ** np.arange(n) * (1 + 0.01 * rng.uniform(-1, 1, size=n))
    u = rng.normal(size=(3, n)); u /= np.sqrt((u ** 2).sum(0))
    pos = rad * u
    pos = pos[:, rng.permutation(n)]
    mass = rng.uniform(0.5, 1.5, size=n) / n
    dacc, dpot = _direct_sum(pos, mass)
    ratio = 0.5 * 1.03
    lmaxes = (2, 6, 12, 24, 40, 48)
    errs = []
    for lmax in lmaxes:
        acc, pot = oracle.mex_force(pos, mass, lmax)
        ep = (np.abs(pot - dpot) / np.abs(dpot)).max()
        ea = (np.sqrt(((acc - dacc) ** 2).sum(0)) / np.sqrt((dacc ** 2).sum(0))).max()
        errs.append((ep, ea))
        assert ep < 5 * ratio ** (lmax + 1) + 1e-13
        assert ea < 5 * (lmax + 2) * ratio ** (lmax + 1) + 1e-12
    assert errs[-1][0] < 1e-12 and errs[-1][1] < 1e-11
    assert errs[0][0] > 1e-3      # and the low-order truncation really is far from Newton


def test_spherical_symmetry_only_Q00():
    # in a spherically symmetric system only Q_00 is nonzero: on (quadrature-)uniform shells the
    # l>0 terms vanish, so lmax=6 reproduces lmax=0
    xc, wc = np.polynomial.legendre.leggauss(8)
    nphi = 16
    ph = (np.arange(nphi) + 0.5) * 2 * math.pi / nphi
    pts, ms = [], []
    for R in (0.5, 1.0, 2.0):
        for x, w in zip(xc, wc):
            s = math.sqrt(1 - x * x)
            for p in ph:
                pts.append([R * s * math.cos(p), R * s * math.sin(p), R * x])
                ms.append(w / nphi)
    pos = np.array(pts).T; mass = np.array(ms)
    # a test particle far outside feels M/r^2 exactly; one inside the innermost shell feels nothing
    pos = np.concatenate([pos, [[7.0], [1.0], [2.0]], [[0.1], [0.05], [-0.02]]], axis=1)
    mass = np.concatenate([mass, [1e-12, 1e-12]])
    a6, p6 = oracle.mex_force(pos, mass, 6)
    M = mass[:-2].sum()
    ro = np.sqrt((pos[:, -2] ** 2).sum())
    assert np.allclose(a6[:, -2], -M * pos[:, -2] / ro ** 3, rtol=1e-12)
    assert np.abs(a6[:, -1]).max() < 1e-12 * M / 0.25


def test_P14_mex_matches_scf_with_large_nmax():
    # eq. (19): MEX == SCF with nmax -> infinity, same lmax.  Loose: SCF includes the self term
    # and a finite nmax; this pins consistent sign/units between the two halves.
    pos, mass = W.particles("hernquist", 4000, seed=1)
    lmax = 2
    am, pm = oracle.mex_force(pos, mass, lmax)
    A, B = oracle.scf_coeffs(pos, mass, 24, lmax)
    asf, ps = oracle.scf_force(pos, 24, lmax, A, B)
    r = np.sqrt((pos ** 2).sum(0))
    sel = (r > 0.3) & (r < 10)
    assert np.median(np.abs(ps[sel] - pm[sel]) / np.abs(pm[sel])) < 2e-2
    arm = (am * pos).sum(0) / r; ars = (asf * pos).sum(0) / r
    assert np.median(np.abs(ars[sel] - arm[sel]) / np.abs(arm[sel])) < 0.1


def test_mex_empty_interior_and_two_particles():
    # degenerate cases: N=1 feels nothing; N=2 is the truncated two-body series
    a, p = oracle.mex_force(np.array([[1.0], [2.0], [3.0]]), np.array([1.0]), 4)
    assert np.all(a == 0) and p[0] == 0
    pos = np.array([[1.0, 0.0], [0.0, 0.0], [0.0, 3.0]])
    mass = np.array([2.0, 5.0])
    a, p = oracle.mex_force(pos, mass, 40)
    da, dp = _direct_sum(pos, mass)
    assert np.allclose(p, dp, rtol=1e-12) and np.allclose(a, da, rtol=1e-11, atol=1e-13)


@pytest.mark.parametrize("lmax,threads", [(0, 1), (6, 1), (8, 3)])
def test_mex_force_at_is_the_definition_and_matches_the_streaming_sweep(lmax, threads):
    """oracle.mex_force_at evaluates eqs. 11-12 for sampled particles straight from their definition (no sort, no
    carried running sum); the streaming oracle must agree with it on every sampled particle, including tied radii,
    the innermost/outermost particles and on-axis ones.  Also pinned to the pairwise series (P11) directly."""
    rng = np.random.default_rng(5)
    n = 3000
    pos, mass = W.particles("plummer", n, seed=3)
    pos[:, 11] = -pos[:, 10]                    # exact tie: 10 is interior to 11
    pos[:, 12] = [0.0, 0.0, 0.5]
    mass = mass * rng.uniform(0.5, 1.5, size=n)
    acc, pot, perm = oracle.mex_force(pos, mass, lmax, return_perm=True)
    idx = np.unique(np.concatenate([[10, 11, 12, perm[0], perm[1], perm[-1], perm[-2]], rng.integers(0, n, 40)]))
    rng.shuffle(idx)                            # sample order must not matter
    acc_s, pot_s = oracle.mex_force_at(pos, mass, lmax, idx, threads=threads)
    assert np.allclose(pot_s, pot[idx], rtol=1e-13, atol=0)
    assert np.allclose(acc_s, acc[:, idx], rtol=1e-12, atol=1e-13 * np.abs(acc).max())
    rank = np.empty(n, dtype=np.int64); rank[perm] = np.arange(n)
    for s in (0, 1, 2):
        i = int(idx[s])
        ref = _pairwise_series_potential(pos[:, i], i, pos, mass, rank, lmax)
        assert pot_s[s] == pytest.approx(float(ref), rel=1e-12)
    with pytest.raises(ValueError):
        oracle.mex_force_at(pos, mass, lmax, [1, 1])
