"""Error metrics of the GPU-vs-oracle parity tests (DESIGN.md "Readings" G13).

north_star: "max relative error of 1e-10 for fp64 coefficients, potentials and accelerations".
  scalars (A, B, pot):  max_i |x_i - ref_i| / max(|ref_i|, floor * max_j |ref_j|),  floor = 1e-6
                        (coefficients that are pure Monte-Carlo noise around zero are measured against the
                        table's scale, not against themselves)
  vectors (acc):        max_i ||a_i - ref_i|| / ||ref_i||
"""
import numpy as np

TOL = 1e-10          # north_star tolerance, fp64
FLOOR = 1e-6


def rel_err_scalar(x, ref, floor=FLOOR):
    x = np.asarray(x, dtype=np.float64)
    ref = np.asarray(ref, dtype=np.float64)
    scale = np.maximum(np.abs(ref), floor * np.max(np.abs(ref)))
    with np.errstate(divide="ignore", invalid="ignore"):
        e = np.where(scale > 0.0, np.abs(x - ref) / scale, np.where(x == ref, 0.0, np.inf))
    return float(np.max(e))


def rel_err_vector(a, ref):
    """a, ref: (3, N)."""
    a = np.asarray(a, dtype=np.float64)
    ref = np.asarray(ref, dtype=np.float64)
    num = np.sqrt(np.sum((a - ref) ** 2, axis=0))
    den = np.sqrt(np.sum(ref ** 2, axis=0))
    with np.errstate(divide="ignore", invalid="ignore"):
        e = np.where(den > 0.0, num / den, np.where(num == 0.0, 0.0, np.inf))   # 0 vs 0 (e.g. innermost particle, lmax=0) agrees
    return float(np.max(e))
