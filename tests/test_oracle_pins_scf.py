"""Pins P3-P9 for the SCF half of the oracle.  None of the expected values below
comes from the oracle itself or from the CUDA path: they are the Poisson equation, exact quadrature,
the analytic Hernquist model, the spherical-harmonic addition theorem and finite differences.  CPU only."""
import math

import numpy as np
import pytest
from scipy import special

import oracle
from paper_1406_4254_b200 import workloads as W

NMAX, LMAX = 10, 6


def test_I00_and_Atilde00():
    # zeroth basis pair is the Hernquist model: I_00 = -1/3, A~_00 = -12 pi
    assert oracle.I_nl(0, 0) == pytest.approx(-1.0 / 3.0, rel=1e-15)
    assert oracle.Atilde_nl(0, 0) == pytest.approx(-12.0 * math.pi, rel=1e-15)
    assert oracle.K_nl(0, 0) == 1.0


def test_zeroth_pair_is_hernquist():
    # Phi~_00 = -1/(1+r), rho~_00 = 1/(2 pi r (1+r)^3): the Hernquist (1990) pair with M=1, a=1
    for r in (1e-4, 0.3, 1.0, 7.0, 300.0):
        phi, dphi = oracle.radial(0, 0, r)
        assert phi[0, 0] == pytest.approx(-1.0 / (1.0 + r), rel=1e-15)
        assert dphi[0, 0] == pytest.approx(1.0 / (1.0 + r) ** 2, rel=1e-14)
        assert oracle.density(0, 0, r)[0, 0] == pytest.approx(1.0 / (2 * math.pi * r * (1 + r) ** 3), rel=1e-14)


def test_P3_radial_poisson_identity():
    # Phi'' + 2 Phi'/r - l(l+1) Phi/r^2 = 4 pi rho  for every (n,l)   ("related via the Poisson equation")
    nmax, lmax = 12, 8
    for r in (0.05, 0.4, 1.0, 2.5, 20.0):
        h = 1e-5 * r
        phi, dphi = oracle.radial(nmax, lmax, r)
        pp, dpp = oracle.radial(nmax, lmax, r + h)
        pm, dpm = oracle.radial(nmax, lmax, r - h)
        rho = oracle.density(nmax, lmax, r)
        # the analytic derivative agrees with a central difference of Phi
        fd1 = (pp - pm) / (2 * h)
        assert np.allclose(dphi, fd1, rtol=1e-7, atol=1e-9 * np.abs(dphi).max())
        d2 = (dpp - dpm) / (2 * h)          # second derivative from the analytic first derivative
        ll = (np.arange(lmax + 1) * (np.arange(lmax + 1) + 1))[:, None]
        lhs = d2 + 2 * dphi / r - ll * phi / r ** 2
        scale = np.abs(d2) + np.abs(2 * dphi / r) + np.abs(ll * phi / r ** 2) + 1e-300
        assert np.all(np.abs(lhs - 4 * math.pi * rho) <= 1e-7 * scale)


def _radial_quadrature(nq):
    x, w = np.polynomial.legendre.leggauss(nq)      # xi in (-1,1); r = (1+xi)/(1-xi); r^2 dr = 2 (1+xi)^2/(1-xi)^4 dxi
    r = (1 + x) / (1 - x)
    jac = 2 * (1 + x) ** 2 / (1 - x) ** 4
    return r, w * jac


def test_P4_biorthogonality_integral_and_Inl():
    # int_0^inf 4 pi rho~_nl Phi~_n'l r^2 dr = I_nl delta_nn'.  In xi the integrand is a polynomial
    # ((1-xi^2)^(2l+1) C_n C_n'), so Gauss-Legendre with enough nodes is exact.
    nmax, lmax = 12, 8
    r, wr = _radial_quadrature(40)
    phi = np.array([oracle.radial(nmax, lmax, ri)[0] for ri in r])      # (nq, l, n)
    rho = np.array([oracle.density(nmax, lmax, ri) for ri in r])
    for l in range(lmax + 1):
        G = 4 * math.pi * np.einsum("q,qn,qm->nm", wr, rho[:, l, :], phi[:, l, :])
        for n in range(nmax + 1):
            I = oracle.I_nl(n, l)
            assert G[n, n] == pytest.approx(I, rel=1e-12)
            assert oracle.Atilde_nl(n, l) == pytest.approx(4 * math.pi / G[n, n], rel=1e-12)
            off = np.delete(G[n], n)
            assert np.all(np.abs(off) <= 1e-12 * abs(I) * (1 + np.abs(np.delete(np.diag(G), n)) / abs(I)))


def test_P5_hernquist_sample_closed_form(oracle_mod):
    # Config-1 sample (equal masses, truncated at r<=300): E[A_000] = 3 E[1/(1+r)] = 303/301,
    # sigma = 0.7048/sqrt(N); other coefficients vanish within noise; pot_i ~ -1/(1+r_i).
    n = 10_000
    pos, mass = W.config_particles(1)
    A, B = oracle.scf_coeffs(pos, mass, NMAX, LMAX)
    L = oracle.num_lm(LMAX)
    assert A[0] == pytest.approx(303.0 / 301.0, abs=4 * 0.7048 / math.sqrt(n))
    # the exact sample value of A_000 from its definition: A~_00 N_00 sum m (-1/(1+r)) = 3 sum m/(1+r)
    r = np.sqrt((pos ** 2).sum(0))
    assert A[0] == pytest.approx(3.0 * math.fsum(mass / (1.0 + r)), rel=1e-13)
    assert np.all(B.reshape(NMAX + 1, L)[:, [oracle.lm_index(l, 0) for l in range(LMAX + 1)]] == 0.0)
    # every other coefficient has zero expectation for a spherical Hernquist sample (biorthogonality in n, isotropy in
    # l,m); its standard error follows from the per-particle terms.  A wrong sign / index / recurrence coefficient in a
    # basis function shows up as a many-sigma mean.
    rad = np.array([oracle.radial(NMAX, LMAX, ri)[0] for ri in r])                       # (N, l, n)
    geo = [oracle.legendre(LMAX, z / ri, math.sqrt(x * x + y * y) / ri)[0] for x, y, z, ri in zip(*pos, r)]
    P = np.array(geo)                                                                    # (N, L)
    phi = np.arctan2(pos[1], pos[0])
    zmax = 0.0
    for l in range(LMAX + 1):
        for m in range(l + 1):
            for nn in range(NMAX + 1):
                if (nn, l, m) == (0, 0, 0):
                    continue
                norm = oracle.Atilde_nl(nn, l) * oracle.N_lm(l, m)
                g = rad[:, l, nn] * P[:, oracle.lm_index(l, m)]
                i = nn * L + oracle.lm_index(l, m)
                se = abs(norm) * np.std(g * np.cos(m * phi)) / math.sqrt(n)
                zmax = max(zmax, abs(A[i]) / se)
                if m > 0:
                    se = abs(norm) * np.std(g * np.sin(m * phi)) / math.sqrt(n)
                    zmax = max(zmax, abs(B[i]) / se)
    assert zmax < 5.5
    acc, pot = oracle.scf_force(pos, NMAX, LMAX, A, B)
    exact = -1.0 / (1.0 + r)
    assert np.median(np.abs(pot - exact) / np.abs(exact)) < 0.05
    # radial acceleration of the Hernquist model: -1/(1+r)^2
    ar = (acc * pos).sum(0) / r
    assert np.median(np.abs(ar + 1.0 / (1.0 + r) ** 2) * (1 + r) ** 2) < 0.1


def test_P5_exact_spherical_model_from_monopole_coefficient():
    # With A_000 = 1 and everything else 0 the SCF field IS the Hernquist model: Phi = -1/(1+r), a = -r_hat/(1+r)^2
    pos, _ = W.particles("hernquist", 500, seed=3)
    T = (NMAX + 1) * oracle.num_lm(LMAX)
    A = np.zeros(T); B = np.zeros(T); A[0] = 1.0
    acc, pot = oracle.scf_force(pos, NMAX, LMAX, A, B)
    r = np.sqrt((pos ** 2).sum(0))
    assert np.allclose(pot, -1.0 / (1.0 + r), rtol=1e-14)
    assert np.allclose(acc, -pos / r / (1.0 + r) ** 2, rtol=1e-13, atol=1e-16)


@pytest.mark.parametrize("target", [(0, 0, 0, "c"), (3, 2, 1, "c"), (3, 2, 1, "s"), (5, 4, 4, "s"), (2, 3, 0, "c"), (7, 6, 3, "c")])
def test_P6_biorthogonality_end_to_end(target):
    # A density equal to ONE basis pair, rho = rho~_n'l'(r) P_l'm'(cos th) {cos,sin}(m' phi), represented by signed
    # point masses on a tensor quadrature grid, returns that single coefficient = 1 and all others = 0
    # (north_star "biorthogonality"; fixes A~_nl N_lm, the table layout and the cos/sin split end to end).
    nmax, lmax = 7, 6
    n0, l0, m0, cs = target
    r, wr = _radial_quadrature(32)
    xc, wc = np.polynomial.legendre.leggauss(16)
    nphi = 16
    ph = (np.arange(nphi) + 0.5) * 2 * math.pi / nphi
    R, Cc, Ph = np.meshgrid(r, xc, ph, indexing="ij")
    Wt = wr[:, None, None] * wc[None, :, None] * (2 * math.pi / nphi) * np.ones_like(Ph)
    rho_r = np.array([oracle.density(nmax, lmax, ri)[l0, n0] for ri in r])
    plm = np.array([oracle.legendre(lmax, x, math.sqrt(1 - x * x))[0][oracle.lm_index(l0, m0)] for x in xc])
    ang = np.cos(m0 * Ph) if cs == "c" else np.sin(m0 * Ph)
    mass = (rho_r[:, None, None] * plm[None, :, None] * ang * Wt).ravel()
    St = np.sqrt(1 - Cc ** 2)
    pos = np.stack([(R * St * np.cos(Ph)).ravel(), (R * St * np.sin(Ph)).ravel(), (R * Cc).ravel()])
    A, B = oracle.scf_coeffs(pos, mass, nmax, lmax)
    L = oracle.num_lm(lmax)
    idx = n0 * L + oracle.lm_index(l0, m0)
    expA = np.zeros_like(A); expB = np.zeros_like(B)
    (expA if cs == "c" else expB)[idx] = 1.0
    assert np.allclose(A, expA, rtol=0, atol=1e-11)
    assert np.allclose(B, expB, rtol=0, atol=1e-11)


def test_P7_pairwise_addition_theorem_identity():
    # Phi_i = sum_j m_j sum_{n,l} (2l+1)/I_nl Phi~_nl(r_i) Phi~_nl(r_j) P_l(cos gamma_ij), j = i included.
    # The angular part here is scipy's Legendre P_l of the pair angle: independent of the oracle's Y_lm code.
    rng = np.random.default_rng(7)
    n = 48
    pos = rng.normal(size=(3, n)) * np.array([[1.0], [0.7], [0.4]])
    pos[:, 0] = [0.0, 0.0, 0.8]          # an on-axis particle
    pos[:, 1] = [0.0, 0.0, -1.3]
    mass = rng.uniform(0.5, 1.5, size=n) / n
    A, B = oracle.scf_coeffs(pos, mass, NMAX, LMAX)
    _, pot = oracle.scf_force(pos, NMAX, LMAX, A, B)
    r = np.sqrt((pos ** 2).sum(0))
    rad = np.array([oracle.radial(NMAX, LMAX, ri)[0] for ri in r])    # (n, l, nn)
    cosg = np.clip((pos.T @ pos) / np.outer(r, r), -1, 1)
    ref = np.zeros(n)
    for l in range(LMAX + 1):
        pl = special.eval_legendre(l, cosg)
        for nn in range(NMAX + 1):
            ref += (2 * l + 1) / oracle.I_nl(nn, l) * rad[:, l, nn] * ((pl * rad[None, :, l, nn]) @ mass)
    assert np.allclose(pot, ref, rtol=1e-12, atol=1e-13 * np.abs(ref).max())


def test_P8_acceleration_is_minus_gradient_of_potential():
    rng = np.random.default_rng(11)
    n = 40
    src, mass = W.particles("hernquist", 2000, seed=5, axes=(1.0, 0.8, 0.6))
    A, B = oracle.scf_coeffs(src, mass, NMAX, LMAX)
    pts = rng.normal(size=(3, n)) * 1.5
    pts[:, 0] = [1e-3, 2e-3, 0.9]        # close to the z axis
    pts[:, 1] = [0.0, 0.0, 0.5]          # on the axis
    acc, _ = oracle.scf_force(pts, NMAX, LMAX, A, B)
    h = 1e-5
    for d in range(3):
        e = np.zeros((3, 1)); e[d] = h
        _, pp = oracle.scf_force(pts + e, NMAX, LMAX, A, B)
        _, pm = oracle.scf_force(pts - e, NMAX, LMAX, A, B)
        _, pp2 = oracle.scf_force(pts + 2 * e, NMAX, LMAX, A, B)
        _, pm2 = oracle.scf_force(pts - 2 * e, NMAX, LMAX, A, B)
        grad = (8 * (pp - pm) - (pp2 - pm2)) / (12 * h)        # 4th-order central difference
        assert np.allclose(acc[d], -grad, rtol=1e-7, atol=1e-8 * np.abs(acc).max())


def test_P9_symmetries():
    rng = np.random.default_rng(3)
    half = rng.normal(size=(3, 100))
    L = oracle.num_lm(LMAX)
    lm = [(l, m) for l in range(LMAX + 1) for m in range(l + 1)]
    # point-mirrored set: odd-l coefficients cancel ("odd terms are in principle zero")
    pos = np.concatenate([half, -half], axis=1)
    mass = np.full(200, 1 / 200)
    A, B = oracle.scf_coeffs(pos, mass, NMAX, LMAX)
    A2, B2 = A.reshape(NMAX + 1, L), B.reshape(NMAX + 1, L)
    odd = [oracle.lm_index(l, m) for l, m in lm if l % 2 == 1]
    assert np.abs(A2[:, odd]).max() < 1e-13 and np.abs(B2[:, odd]).max() < 1e-13
    assert np.abs(A2[:, [oracle.lm_index(2, 0)]]).max() > 1e-3
    # axisymmetric rings ("Q_lm = 0 for all |m| > 0"): 16 equal masses per ring, m = 1..6 vanish
    k = 16
    ph = np.arange(k) * 2 * math.pi / k
    rings = []
    for R, z in ((0.5, 0.2), (1.5, -0.7), (3.0, 0.1)):
        rings.append(np.stack([R * np.cos(ph), R * np.sin(ph), np.full(k, z)]))
    pos = np.concatenate(rings, axis=1)
    mass = np.full(pos.shape[1], 1 / pos.shape[1])
    A, B = oracle.scf_coeffs(pos, mass, NMAX, LMAX)
    A2, B2 = A.reshape(NMAX + 1, L), B.reshape(NMAX + 1, L)
    nz = [oracle.lm_index(l, m) for l, m in lm if m != 0]
    assert np.abs(A2[:, nz]).max() < 1e-13 and np.abs(B2[:, nz]).max() < 1e-13
    assert np.abs(A2[:, oracle.lm_index(2, 0)]).max() > 1e-3


def test_thread_count_does_not_change_coefficients_beyond_rounding():
    pos, mass = W.config_particles(1, n=3000)
    A1, B1 = oracle.scf_coeffs(pos, mass, NMAX, LMAX, threads=1)
    A4, B4 = oracle.scf_coeffs(pos, mass, NMAX, LMAX, threads=4)
    assert np.allclose(A1, A4, rtol=0, atol=1e-15) and np.allclose(B1, B4, rtol=0, atol=1e-15)
