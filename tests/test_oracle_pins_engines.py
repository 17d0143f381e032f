"""Pins P1, P2: the oracle's recurrence engines against closed forms, library
routines and identities that do not come from the oracle itself.  CPU only."""
import math
import os

import mpmath as mp
import numpy as np
import pytest
from scipy import special

import oracle

GOLDEN = os.path.join(os.path.dirname(__file__), "golden", "paper_counts.txt")


def test_paper_counts_golden():
    # sizes the paper prints.
    for line in open(GOLDEN):
        if line.startswith("#") or not line.strip():
            continue
        kind, nmax, lmax, value = line.split()[:4]
        nmax, lmax, value = int(nmax), int(lmax), int(value)
        if kind == "scf_complex_coeffs":
            assert (nmax + 1) * oracle.num_lm(lmax) == value
        elif kind == "mex_complex_pairs":
            assert oracle.num_lm(lmax) == value
        elif kind == "scf_table_bytes":
            assert (nmax + 1) * oracle.num_lm(lmax) * 16 == value
    assert oracle.lm_index(6, 6) == oracle.num_lm(6) - 1


# ------------------------------------------------------------------ P1: Gegenbauer engine
XIS = [-0.999, -0.7, -0.2, 0.0, 0.31, 0.85, 0.9999]
ALPHAS = [1.5, 3.5, 5.5, 13.5, 21.5]


def test_gegenbauer_closed_forms():
    for a in ALPHAS:
        for x in XIS:
            c, d = oracle.gegenbauer(3, a, x)
            assert c[0] == 1.0 and d[0] == 0.0
            assert c[1] == pytest.approx(2 * a * x, rel=1e-15)
            assert c[2] == pytest.approx(2 * a * (a + 1) * x * x - a, rel=1e-13, abs=1e-13)
            assert c[3] == pytest.approx(4.0 / 3.0 * a * (a + 1) * (a + 2) * x ** 3 - 2 * a * (a + 1) * x, rel=1e-13, abs=1e-12)


def test_gegenbauer_value_at_one_and_parity():
    for a in ALPHAS:
        c, _ = oracle.gegenbauer(20, a, 1.0)
        cm, _ = oracle.gegenbauer(20, a, -1.0)
        for n in range(21):
            exact = float(mp.gamma(n + 2 * a) / (mp.factorial(n) * mp.gamma(2 * a)))
            assert c[n] == pytest.approx(exact, rel=1e-13)
            assert cm[n] == pytest.approx((-1) ** n * exact, rel=1e-13)
        cp, _ = oracle.gegenbauer(20, a, 0.37)
        cn, _ = oracle.gegenbauer(20, a, -0.37)
        assert np.allclose(cn, cp * (-1.0) ** np.arange(21), rtol=1e-14, atol=0)


def test_gegenbauer_special_alphas():
    # alpha = 1/2 -> Legendre P_n ; alpha = 1 -> Chebyshev U_n(cos t) = sin((n+1)t)/sin t
    for x in XIS:
        c, _ = oracle.gegenbauer(12, 0.5, x)
        assert np.allclose(c, special.eval_legendre(np.arange(13), x), rtol=1e-13, atol=1e-14)
        t = math.acos(x)
        c, _ = oracle.gegenbauer(12, 1.0, x)
        u = np.sin((np.arange(13) + 1) * t) / math.sin(t)
        assert np.allclose(c, u, rtol=1e-10, atol=1e-10)


def _gegenbauer_explicit(n, a, x):
    """C_n^(a)(x) = sum_k (-1)^k Gamma(n-k+a) / (Gamma(a) k! (n-2k)!) (2x)^(n-2k), in 40 digits."""
    if n < 0:
        return mp.mpf(0)
    a, x = mp.mpf(a), mp.mpf(x)
    return sum((-1) ** k * mp.gamma(n - k + a) / (mp.gamma(a) * mp.factorial(k) * mp.factorial(n - 2 * k)) * (2 * x) ** (n - 2 * k)
               for k in range(n // 2 + 1))


def test_gegenbauer_vs_libraries_and_derivative():
    mp.mp.dps = 40
    for a in ALPHAS:
        for x in XIS:
            c, d = oracle.gegenbauer(20, a, x)
            ref = special.eval_gegenbauer(np.arange(21), a, x)
            scale = np.maximum(np.abs(ref), np.abs(ref).max() * 1e-3)
            assert np.all(np.abs(c - ref) <= 2e-13 * scale)
            for n in (0, 1, 2, 5, 11, 20):
                # tolerance relative to the polynomial's envelope on [-1,1], C_n^(a)(1)
                exact = _gegenbauer_explicit(n, a, x)
                assert abs(c[n] - exact) <= 1e-13 * max(abs(exact), 1e-2 * _gegenbauer_explicit(n, a, 1))
                # C'_n^(a) = 2a C_{n-1}^(a+1)
                dex = 2 * a * _gegenbauer_explicit(n - 1, a + 1, x)
                assert abs(d[n] - dex) <= 1e-13 * max(abs(dex), 1e-2 * 2 * a * _gegenbauer_explicit(n - 1, a + 1, 1))


def test_gegenbauer_generating_function_and_ode():
    # (1 - 2 x t + t^2)^-a = sum_n C_n(x) t^n
    a, x, t = 3.5, 0.43, 0.2
    c, d = oracle.gegenbauer(60, a, x)
    s = sum(c[n] * t ** n for n in range(61))
    assert s == pytest.approx((1 - 2 * x * t + t * t) ** (-a), rel=1e-13)
    # ODE (1-x^2) y'' - (2a+1) x y' + n(n+2a) y = 0, y'' from C'_n = 2a C_{n-1}^(a+1) twice (via oracle at a+1)
    for a in (1.5, 5.5):
        for x in (-0.6, 0.2, 0.9):
            c, d = oracle.gegenbauer(12, a, x)
            c1, d1 = oracle.gegenbauer(12, a + 1, x)
            for n in range(2, 13):
                ypp = 2 * a * d1[n - 1]
                res = (1 - x * x) * ypp - (2 * a + 1) * x * d[n] + n * (n + 2 * a) * c[n]
                assert abs(res) <= 1e-11 * (abs(n * (n + 2 * a) * c[n]) + abs(ypp) + 1)


# ------------------------------------------------------------------ P2: Legendre engine
THETAS = [1e-4, 0.05, 0.7, math.pi / 2, 2.3, math.pi - 1e-4]


def test_legendre_closed_forms():
    for th in THETAS:
        c, s = math.cos(th), math.sin(th)
        p, d, u = oracle.legendre(3, c, s)
        i = oracle.lm_index
        exp = {(0, 0): 1, (1, 0): c, (1, 1): s, (2, 0): 0.5 * (3 * c * c - 1), (2, 1): 3 * c * s, (2, 2): 3 * s * s,
               (3, 0): 0.5 * (5 * c ** 3 - 3 * c), (3, 1): 1.5 * (5 * c * c - 1) * s, (3, 2): 15 * c * s * s, (3, 3): 15 * s ** 3}
        for (l, m), v in exp.items():
            assert p[i(l, m)] == pytest.approx(v, rel=1e-14, abs=1e-300)
        dexp = {(0, 0): 0, (1, 0): -s, (1, 1): c, (2, 0): -3 * c * s, (2, 1): 3 * (c * c - s * s), (2, 2): 6 * s * c,
                (3, 3): 45 * s * s * c}
        for (l, m), v in dexp.items():
            assert d[i(l, m)] == pytest.approx(v, rel=1e-13, abs=1e-18)
        # U = P / sin, regular on the axis: only m=1 survives there
        assert u[i(1, 1)] == 1.0
        assert u[i(2, 1)] == pytest.approx(3 * c, rel=1e-15)
        assert u[i(3, 3)] == pytest.approx(15 * s * s, rel=1e-14, abs=1e-300)


def _legendre_poly_derivative(l, k, x):
    """d^k/dx^k P_l(x) from the explicit power series P_l(x) = 2^-l sum_j (-1)^j C(l,j) C(2l-2j,l) x^(l-2j), in mpmath."""
    tot = mp.mpf(0)
    for j in range(l // 2 + 1):
        e = l - 2 * j
        if e < k:
            continue
        tot += (-1) ** j * mp.binomial(l, j) * mp.binomial(2 * l - 2 * j, l) * mp.ff(e, k) * x ** (e - k)
    return tot / mp.mpf(2) ** l


def test_legendre_vs_scipy_and_mpmath_near_poles():
    # exact reference: P_l^m(cos t) = sin^m t D^m P_l(x)  (no Condon-Shortley phase), and by the chain rule
    # dP_l^m/dt = m cos t sin^(m-1) t D^m P_l - sin^(m+1) t D^(m+1) P_l, evaluated in 30 digits from theta itself
    mp.mp.dps = 30
    lmax = 10
    for th in THETAS:
        c, s = math.cos(th), math.sin(th)
        p, d, u = oracle.legendre(lmax, c, s)
        tq = mp.mpf(th)
        x, sq = mp.cos(tq), mp.sin(tq)
        for l in range(lmax + 1):
            for m in range(l + 1):
                j = oracle.lm_index(l, m)
                dm, dm1 = _legendre_poly_derivative(l, m, x), _legendre_poly_derivative(l, m + 1, x)
                ref = sq ** m * dm
                # relative accuracy, except next to an interior zero where the scale is the function's envelope
                # sqrt((l+m)!/(l-m)!) sin^m (so the poles, where P_lm -> 0 like sin^m, are still tested relatively)
                env = mp.sqrt(mp.factorial(l + m) / mp.factorial(l - m)) * sq ** m
                tol = 2e-14 * max(abs(ref), env * mp.mpf("0.05"))
                assert abs(p[j] - ref) <= tol, (th, l, m)
                if m >= 1:
                    assert abs(u[j] - ref / sq) <= tol / sq, (th, l, m)
                dref = (m * x * sq ** (m - 1) * dm if m >= 1 else 0) - sq ** (m + 1) * dm1
                denv = mp.sqrt(mp.factorial(l + m) / mp.factorial(l - m)) * max(l, 1) * (sq ** max(m - 1, 0))
                assert abs(d[j] - dref) <= 1e-13 * max(abs(dref), denv * mp.mpf("0.05")), (th, l, m)
        if 0.01 < th < 3.1:   # scipy's lpmv carries the Condon-Shortley phase; fine away from the poles
            for l in range(lmax + 1):
                for m in range(l + 1):
                    ref = (-1) ** m * special.lpmv(m, l, c)
                    assert p[oracle.lm_index(l, m)] == pytest.approx(ref, rel=1e-12, abs=1e-12 * math.sqrt(math.factorial(l + m) / math.factorial(l - m)))


def test_addition_theorem_and_normalisation():
    # sum_{m>=0} N_lm P_lm^2 = (2l+1)/4pi at any theta  (north_star; fixes N_lm and the (2-delta_m0) folding)
    lmax = 10
    for th in THETAS:
        p, _, _ = oracle.legendre(lmax, math.cos(th), math.sin(th))
        for l in range(lmax + 1):
            s = sum(oracle.N_lm(l, m) * p[oracle.lm_index(l, m)] ** 2 for m in range(l + 1))
            assert s == pytest.approx((2 * l + 1) / (4 * math.pi), rel=1e-13)
    for l in range(lmax + 1):
        for m in range(l + 1):
            w = (1 if m == 0 else 2) * math.factorial(l - m) / math.factorial(l + m)
            assert oracle.w_lm(l, m) == pytest.approx(w, rel=1e-15)
            assert oracle.N_lm(l, m) == pytest.approx(w * (2 * l + 1) / (4 * math.pi), rel=1e-15)


def test_real_harmonics_orthonormal_on_quadrature():
    # Gauss-Legendre in cos(theta) x uniform phi: int N_lm P_lm P_l'm {cos,sin}^2 = delta_ll'
    lmax, nq = 8, 24
    x, wq = np.polynomial.legendre.leggauss(nq)
    tab = np.array([oracle.legendre(lmax, xi, math.sqrt(1 - xi * xi))[0] for xi in x])   # (nq, L)
    for m in range(lmax + 1):
        phi_int = 2 * math.pi if m == 0 else math.pi    # int cos^2(m phi) dphi
        for l in range(m, lmax + 1):
            for l2 in range(m, lmax + 1):
                integ = np.sum(wq * tab[:, oracle.lm_index(l, m)] * tab[:, oracle.lm_index(l2, m)]) * phi_int
                # N_lm folds +-m into m >= 0, so  N_lm int P_lm^2 dcos int cos^2(m phi) dphi = 1 for every m
                val = integ * oracle.N_lm(l, m)
                expect = 1.0 if l == l2 else 0.0
                if l != l2:
                    assert abs(val) < 1e-12
                else:
                    assert val == pytest.approx(expect, rel=1e-12)


def test_eq24_recurrence_is_unstable_near_axis():
    # Negative pin (reading G3): the paper's m-recurrence
    #   P_lm = -2(m-1) cot(theta) P_{l,m-1} - (l+m-1)(l-m+2) P_{l,m-2}   (CS-phase convention)
    # is exact mid-range and loses all digits near the pole, which is why the oracle does not use it.
    def eq24(l, th):
        c, s = math.cos(th), math.sin(th)
        out = [special.eval_legendre(l, c), special.lpmv(1, l, c)]
        for m in range(2, l + 1):
            out.append(-2 * (m - 1) * (c / s) * out[m - 1] - (l + m - 1) * (l - m + 2) * out[m - 2])
        return out
    l = 6
    mid = eq24(l, 0.7)
    p, _, _ = oracle.legendre(l, math.cos(0.7), math.sin(0.7))
    for m in range(l + 1):
        assert mid[m] == pytest.approx((-1) ** m * p[oracle.lm_index(l, m)], rel=1e-10)
    near = eq24(l, 1e-4)
    p, _, _ = oracle.legendre(l, math.cos(1e-4), math.sin(1e-4))
    rel = [abs(near[m] - (-1) ** m * p[oracle.lm_index(l, m)]) / abs(p[oracle.lm_index(l, m)]) for m in range(3, l + 1)]
    assert max(rel) > 1e-3
