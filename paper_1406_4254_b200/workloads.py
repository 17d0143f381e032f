"""Seeded synthetic particle sets for the ETICS hot path.

This module is the ONLY code shared by the CPU oracle (oracle/) and the CUDA path: it produces
plain numpy buffers and contains none of the method's arithmetic (no basis functions, no sums).
It stands in for the paper's workloads: Fig. 5 used unspecified particle sets and states that
the timing "only depends on the number of particles (and expansion cutoffs) and not on their
spatial distribution" (§3.4); §4.2 used an N=10^6 Hernquist sphere with a=1
(PAPER.md:338).  No public dataset is involved.

Generator: counter-based, particle k depends only on (seed, k):
    h_s = mix64(seed, k, s), s in {0,1,2};  u,v,w = ((h_s >> 11) + 0.5) * 2^-53  in (0,1)
    radius from u by the model's inverse CDF (truncated by scaling u, no rejection loop),
    cos(theta) = 1 - 2 v,  phi = 2 pi w,  masses 1/N.
Layouts match the C ABI (include/etics.h): pos is (3, N) C-contiguous float64 (x | y | z), mass is (N,).
"""
from __future__ import annotations

import numpy as np

_M64 = np.uint64(0xFFFFFFFFFFFFFFFF)


def mix64(seed: int, k: np.ndarray, stream: int) -> np.ndarray:
    """64-bit finaliser-style hash of (seed, k, stream); k is a uint64 array."""
    with np.errstate(over="ignore"):
        z = (k.astype(np.uint64) * np.uint64(0x9E3779B97F4A7C15)
             + np.uint64((seed * 0xD1B54A32D192ED03 + stream * 0x8CB92BA72F3D8DD7 + 0x2545F4914F6CDD1D) & 0xFFFFFFFFFFFFFFFF))
        z ^= z >> np.uint64(30)
        z *= np.uint64(0xBF58476D1CE4E5B9)
        z ^= z >> np.uint64(27)
        z *= np.uint64(0x94D049BB133111EB)
        z ^= z >> np.uint64(31)
        z *= np.uint64(0xD6E8FEB86659FD93)
        z ^= z >> np.uint64(32)
    return z


def uniforms(seed: int, n: int, stream: int, start: int = 0) -> np.ndarray:
    """n uniform deviates in the open interval (0,1), one per particle index start..start+n-1."""
    k = np.arange(start, start + n, dtype=np.uint64)
    h = mix64(seed, k, stream)
    return ((h >> np.uint64(11)).astype(np.float64) + 0.5) * (2.0 ** -53)


HERNQUIST_RMAX = 300.0
PLUMMER_RMAX = 100.0


def _radius(model: str, u: np.ndarray) -> np.ndarray:
    if model == "hernquist":
        # M(<r)/M = r^2/(1+r)^2 = u  =>  r = sqrt(u)/(1-sqrt(u)); truncation r<=300 <=> u <= (300/301)^2
        umax = (HERNQUIST_RMAX / (1.0 + HERNQUIST_RMAX)) ** 2
        s = np.sqrt(u * umax)
        return s / (1.0 - s)
    if model == "plummer":
        # M(<r)/M = r^3/(1+r^2)^(3/2) = u  =>  r = (u^(-2/3)-1)^(-1/2); r<=100 <=> u <= (1e4/10001)^1.5
        umax = (PLUMMER_RMAX ** 2 / (1.0 + PLUMMER_RMAX ** 2)) ** 1.5
        return 1.0 / np.sqrt((u * umax) ** (-2.0 / 3.0) - 1.0)
    raise ValueError(f"unknown model {model!r}")


def particles(model: str, n: int, seed: int = 0, axes=(1.0, 1.0, 1.0), chunk: int = 1 << 22):
    """Return (pos, mass): pos (3,n) float64 C-contiguous, mass (n,) float64 = 1/n.

    model: "hernquist" | "plummer"; axes scales (x,y,z) after spherical sampling
    (config 4's triaxial set uses axes=(1.0, 0.8, 0.6)).
    """
    pos = np.empty((3, n), dtype=np.float64)
    for s in range(0, n, chunk):
        m = min(chunk, n - s)
        r = _radius(model, uniforms(seed, m, 0, s))
        ct = 1.0 - 2.0 * uniforms(seed, m, 1, s)
        st = np.sqrt(np.maximum(0.0, (1.0 - ct) * (1.0 + ct)))
        ph = (2.0 * np.pi) * uniforms(seed, m, 2, s)
        pos[0, s:s + m] = axes[0] * r * st * np.cos(ph)
        pos[1, s:s + m] = axes[1] * r * st * np.sin(ph)
        pos[2, s:s + m] = axes[2] * r * ct
    mass = np.full(n, 1.0 / n, dtype=np.float64)
    return pos, mass


# The five configurations of BASELINE.json ("configs"), by index.
CONFIGS = {
    1: dict(method="scf", model="hernquist", n=10_000, nmax=10, lmax=6, axes=(1.0, 1.0, 1.0)),
    2: dict(method="scf", model="hernquist", n=1_000_000, nmax=10, lmax=6, axes=(1.0, 1.0, 1.0)),
    3: dict(method="mex", model="hernquist", n=1_000_000, lmax=6, axes=(1.0, 1.0, 1.0)),
    4: dict(method="scf", model="hernquist", n=10_000_000, nmax=20, lmax=10, axes=(1.0, 0.8, 0.6)),
    5: dict(method="scf+mex", model="plummer", n=100_000_000, nmax=10, lmax=6, mex_lmax=8, axes=(1.0, 1.0, 1.0)),
}


def config_particles(idx: int, n: int | None = None, seed: int = 0):
    """Particles of BASELINE.json config idx (optionally with a different N for tests)."""
    c = CONFIGS[idx]
    return particles(c["model"], c["n"] if n is None else n, seed=seed, axes=c["axes"])
