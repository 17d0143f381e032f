"""ctypes binding of the CPU oracle (oracle/etics_oracle.cpp).

TEST INFRASTRUCTURE, NOT THE PRODUCT: only tests/, __graft_entry__.smoke() and bench.py's
cpu_baseline / --impl reference legs may import this package.  Nothing here touches CUDA, and the
CUDA package never imports it.  Layouts are those of include/etics.h (pos (3,N) x|y|z, A/B index
n*L + l(l+1)/2 + m).
"""
from __future__ import annotations

import ctypes as C

import numpy as np

from . import build as _build

_lib = None
_dp = C.POINTER(C.c_double)


def lib():
    global _lib
    if _lib is None:
        L = C.CDLL(_build.build())
        L.oracle_K_nl.restype = C.c_double
        L.oracle_I_nl.restype = C.c_double
        L.oracle_Atilde_nl.restype = C.c_double
        L.oracle_N_lm.restype = C.c_double
        L.oracle_w_lm.restype = C.c_double
        for f in (L.oracle_K_nl, L.oracle_I_nl, L.oracle_Atilde_nl, L.oracle_N_lm, L.oracle_w_lm):
            f.argtypes = [C.c_int, C.c_int]
        L.oracle_gegenbauer.argtypes = [C.c_int, C.c_double, C.c_double, _dp, _dp]
        L.oracle_legendre.argtypes = [C.c_int, C.c_double, C.c_double, _dp, _dp, _dp]
        L.oracle_radial.argtypes = [C.c_int, C.c_int, C.c_double, _dp, _dp]
        L.oracle_density.argtypes = [C.c_int, C.c_int, C.c_double, _dp]
        L.oracle_scf_coeffs.argtypes = [_dp, _dp, C.c_longlong, C.c_int, C.c_int, _dp, _dp, C.c_int]
        L.oracle_scf_force.argtypes = [_dp, C.c_longlong, C.c_int, C.c_int, _dp, _dp, _dp, _dp, C.c_int]
        L.oracle_mex_sort.argtypes = [_dp, C.c_longlong, C.POINTER(C.c_ulonglong), C.POINTER(C.c_uint)]
        L.oracle_mex_force.argtypes = [_dp, _dp, C.c_longlong, C.c_int, _dp, _dp, C.POINTER(C.c_uint)]
        L.oracle_mex_force_at.argtypes = [_dp, _dp, C.c_longlong, C.c_int, C.POINTER(C.c_longlong), C.c_int, _dp, _dp, C.c_int]
        L.oracle_num_threads.argtypes = [C.c_int]
        _lib = L
    return _lib


def _p(a):
    return a.ctypes.data_as(_dp)


def _f64(a):
    return np.ascontiguousarray(a, dtype=np.float64)


def num_lm(lmax: int) -> int:
    return (lmax + 1) * (lmax + 2) // 2


def lm_index(l: int, m: int) -> int:
    return l * (l + 1) // 2 + m


def num_threads(threads: int = 0) -> int:
    return lib().oracle_num_threads(threads)


def K_nl(n, l): return lib().oracle_K_nl(n, l)
def I_nl(n, l): return lib().oracle_I_nl(n, l)
def Atilde_nl(n, l): return lib().oracle_Atilde_nl(n, l)
def N_lm(l, m): return lib().oracle_N_lm(l, m)
def w_lm(l, m): return lib().oracle_w_lm(l, m)


def gegenbauer(nmax: int, alpha: float, xi: float):
    c = np.empty(nmax + 1); d = np.empty(nmax + 1)
    lib().oracle_gegenbauer(nmax, alpha, xi, _p(c), _p(d))
    return c, d


def legendre(lmax: int, ct: float, st: float):
    n = num_lm(lmax)
    p = np.empty(n); d = np.empty(n); u = np.empty(n)
    lib().oracle_legendre(lmax, ct, st, _p(p), _p(d), _p(u))
    return p, d, u


def radial(nmax: int, lmax: int, r: float):
    """Phi~_nl(r), dPhi~_nl/dr as arrays [l, n]."""
    a = np.empty((lmax + 1, nmax + 1)); b = np.empty((lmax + 1, nmax + 1))
    lib().oracle_radial(nmax, lmax, r, _p(a), _p(b))
    return a, b


def density(nmax: int, lmax: int, r: float):
    a = np.empty((lmax + 1, nmax + 1))
    lib().oracle_density(nmax, lmax, r, _p(a))
    return a


def scf_coeffs(pos, mass, nmax: int, lmax: int, threads: int = 0):
    pos = _f64(pos); mass = _f64(mass)
    n = mass.shape[0]
    assert pos.shape == (3, n)
    t = (nmax + 1) * num_lm(lmax)
    a = np.empty(t); b = np.empty(t)
    rc = lib().oracle_scf_coeffs(_p(pos), _p(mass), n, nmax, lmax, _p(a), _p(b), threads)
    if rc != 0:
        raise ValueError(f"oracle_scf_coeffs failed: {rc}")
    return a, b


def scf_force(pos, nmax: int, lmax: int, a, b, threads: int = 0):
    pos = _f64(pos); a = _f64(a); b = _f64(b)
    n = pos.shape[1]
    assert pos.shape == (3, n) and a.shape == b.shape == ((nmax + 1) * num_lm(lmax),)
    acc = np.empty((3, n)); pot = np.empty(n)
    rc = lib().oracle_scf_force(_p(pos), n, nmax, lmax, _p(a), _p(b), _p(acc), _p(pot), threads)
    if rc != 0:
        raise ValueError(f"oracle_scf_force failed: {rc}")
    return acc, pot


def mex_sort(pos):
    pos = _f64(pos)
    n = pos.shape[1]
    keys = np.empty(n, dtype=np.uint64); perm = np.empty(n, dtype=np.uint32)
    rc = lib().oracle_mex_sort(_p(pos), n, keys.ctypes.data_as(C.POINTER(C.c_ulonglong)), perm.ctypes.data_as(C.POINTER(C.c_uint)))
    if rc != 0:
        raise ValueError(f"oracle_mex_sort failed: {rc}")
    return keys, perm


def mex_force(pos, mass, lmax: int, return_perm: bool = False):
    pos = _f64(pos); mass = _f64(mass)
    n = mass.shape[0]
    assert pos.shape == (3, n)
    acc = np.empty((3, n)); pot = np.empty(n)
    perm = np.empty(n, dtype=np.uint32)
    rc = lib().oracle_mex_force(_p(pos), _p(mass), n, lmax, _p(acc), _p(pot), perm.ctypes.data_as(C.POINTER(C.c_uint)))
    if rc != 0:
        raise ValueError(f"oracle_mex_force failed: {rc}")
    return (acc, pot, perm) if return_perm else (acc, pot)


def mex_force_at(pos, mass, lmax: int, sample_idx, threads: int = 0):
    """MEX potential/acceleration of the sampled particles straight from eqs. 11-12 (no sort); (3,S), (S)."""
    pos = _f64(pos); mass = _f64(mass)
    n = mass.shape[0]
    assert pos.shape == (3, n)
    idx = np.ascontiguousarray(np.asarray(sample_idx, dtype=np.int64))
    s = idx.shape[0]
    acc = np.empty((3, s)); pot = np.empty(s)
    rc = lib().oracle_mex_force_at(_p(pos), _p(mass), n, lmax, idx.ctypes.data_as(C.POINTER(C.c_longlong)), s,
                                   _p(acc), _p(pot), threads)
    if rc != 0:
        raise ValueError(f"oracle_mex_force_at failed: {rc}")
    return acc, pot


def leapfrog(force, pos, vel, dt: float, nsteps: int):
    """Kick-drift-kick leapfrog of x'' = a(x) (§3.4: the systems are evolved with a leapfrog that calls the
    force routine once per step), written out step by step:
        v += (dt/2) a(x);  x += dt v;  a = force(x);  v += (dt/2) a(x)
    force(pos) -> acc, both (3, N).  Returns (pos, vel, acc) after nsteps steps; the inputs are not modified."""
    x = _f64(pos).copy(); v = _f64(vel).copy()
    a = force(x)
    for _ in range(nsteps):
        v = v + (0.5 * dt) * a
        x = x + dt * v
        a = force(x)
        v = v + (0.5 * dt) * a
    return x, v, a


def scf_acceleration(mass, nmax: int, lmax: int, every: int = 1):
    """force(pos) for leapfrog(): the SCF full force calculation on the particles themselves.  every > 1: "temporal
    softening": the coefficients are recomputed at force evaluations 0, every, 2 every, ... and held in
    between (evaluation 0 is a(x_0), evaluation j the force of step j)."""
    state = {"calls": 0, "AB": None}

    def f(x):
        if state["calls"] % every == 0:
            state["AB"] = scf_coeffs(x, mass, nmax, lmax)
        state["calls"] += 1
        return scf_force(x, nmax, lmax, *state["AB"])[0]
    f.state = state
    return f


def mex_acceleration(mass, lmax: int):
    """force(pos) for leapfrog(): the MEX full force calculation."""
    return lambda x: mex_force(x, mass, lmax)[0]
