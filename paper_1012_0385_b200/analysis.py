"""Host-side post-processing of the records the library returns: the paper's observables.

Nothing here runs on the hot path: the kernels deliver exact integers (sum h, sum h^2 per sample and record time; hop
counts J_A, J_B), and these few numpy lines turn them into what the paper plots -
  * W^2(t, L), Eq. 3 squared, averaged over samples,
  * effective exponents (Eqs. 4-6) and the finite-size-scaling collapse with (alpha, z)
    (Fig. 3; 157-167, Fig. 4),
  * the current density c = (J_A - J_B)/L of the two-lane model and its fluctuation <c^2>(t).
"""
from __future__ import annotations

import numpy as np


def w2_per_sample(L: int, sum_h, sum_h2) -> np.ndarray:
    """W^2 = sum h^2 / L - (sum h / L)^2 per (record, sample) from the exact integer sums; the numerator
    L*sum_h2 - sum_h^2 is formed in Python integers (it can exceed 64 bits), one rounding to double."""
    a = np.asarray(sum_h, dtype=object)
    b = np.asarray(sum_h2, dtype=object)
    num = L * b - a * a
    flat = [float(int(x)) / (float(L) * float(L)) for x in num.ravel()]     # same rounding as the library
    return np.array(flat, dtype=np.float64).reshape(np.shape(num))


def w2_mean(L: int, sum_h, sum_h2) -> np.ndarray:
    """Mean over samples of the per-sample W^2 - not the width of the pooled heights."""
    return w2_per_sample(L, sum_h, sum_h2).mean(axis=-1)


def local_exponents(t, y) -> np.ndarray:
    """d ln y / d ln t between consecutive record times (effective exponent; for y = W^2 - 1/4 this is 2 beta)."""
    t = np.asarray(t, dtype=np.float64)
    y = np.asarray(y, dtype=np.float64)
    return np.diff(np.log(y)) / np.diff(np.log(t))


def growth_exponent(t, w2, t_min=32.0, intrinsic=0.25) -> float:
    """beta from a least-squares line through ln(W^2 - 1/4) vs ln t for t >= t_min (PAPER.md:139 subtracts the
    intrinsic width 1/4 of the zig-zag start)."""
    t = np.asarray(t, dtype=np.float64)
    y = np.asarray(w2, dtype=np.float64) - intrinsic
    sel = t >= t_min
    return 0.5 * float(np.polyfit(np.log(t[sel]), np.log(y[sel]), 1)[0])


def collapse(L, t, w2, alpha: float, z: float, intrinsic=0.25):
    """Family-Vicsek rescaling of one size: (t / L^z, (W^2 - 1/4) / L^(2 alpha)) (Fig. 3b, 4b)."""
    t = np.asarray(t, dtype=np.float64)
    y = np.asarray(w2, dtype=np.float64) - intrinsic
    return t / float(L) ** z, y / float(L) ** (2.0 * alpha)


def collapse_spread(curves, alpha: float, z: float, intrinsic=0.25) -> float:
    """A scalar quality of a collapse: rescale every (L, t, W^2) curve, interpolate them in ln-ln on the common range
    of the rescaled time and return the mean over that range of the relative spread between sizes (0 = perfect)."""
    xs, ys = [], []
    for L, t, w2 in curves:
        x, y = collapse(L, t, w2, alpha, z, intrinsic)
        ok = y > 0
        xs.append(np.log(x[ok]))
        ys.append(np.log(y[ok]))
    lo, hi = max(x.min() for x in xs), min(x.max() for x in xs)
    if not lo < hi:
        raise ValueError("the rescaled curves do not overlap")
    grid = np.linspace(lo, hi, 32)
    vals = np.array([np.interp(grid, x, y) for x, y in zip(xs, ys)])
    return float(np.mean(vals.max(axis=0) - vals.min(axis=0)))


def current_fluctuation(j_a, j_b, L: int):
    """Two-lane model: c = (J_A - J_B)/L per (record, sample); returns (<c>, <c^2>) per record time.
    J_A and J_B are both counted positive by the library: lane A moves right, lane B left."""
    c = (np.asarray(j_a, dtype=np.float64) - np.asarray(j_b, dtype=np.float64)) / float(L)
    return c.mean(axis=-1), (c * c).mean(axis=-1)
