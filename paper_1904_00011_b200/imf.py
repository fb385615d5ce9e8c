"""Host-side IMF weights of an isochrone's mass points (a Salpeter IMF by default, a
Kroupa IMF also implemented; the weights of an isochrone follow the IMF).  Argument
preparation only: the library takes `imf_w[J]`, summing to 1 inside each isochrone (DESIGN.md R-Q2),
whatever produced it.

A point's weight is the integral of the IMF over its mass cell; cells are bounded by the geometric
mid-points of neighbouring masses (the first and last cell end at the first and last mass), the
convention of workloads/synthetic.py.
"""
from __future__ import annotations

import numpy as np

# (upper mass edge of the segment, slope alpha of dN/dm ~ m^-alpha)
SALPETER = ((np.inf, 2.35),)
KROUPA = ((0.08, 0.3), (0.5, 1.3), (np.inf, 2.3))


def _segments(imf):
    """[(m_lo, m_hi, alpha, continuity factor)] of a broken power law, continuous at the breaks."""
    out, lo, c = [], 0.0, 1.0
    for k, (hi, alpha) in enumerate(imf):
        if k > 0:
            c *= lo ** (alpha - imf[k - 1][1])      # c_k lo^-alpha_k = c_{k-1} lo^-alpha_{k-1}
        out.append((lo, hi, alpha, c))
        lo = hi
    return out


def cumulative(m, imf=KROUPA) -> np.ndarray:
    """Integral of the (unnormalised) IMF from 0.01 Msun to m."""
    m = np.atleast_1d(np.asarray(m, dtype=np.float64))
    total = np.zeros_like(m)
    for lo, hi, alpha, c in _segments(imf):
        a = np.clip(m, max(lo, 0.01), hi if np.isfinite(hi) else None)
        b = max(lo, 0.01)
        p = 1.0 - alpha
        total += c * (a ** p - b ** p) / p if p != 0 else c * np.log(a / b)
    return total


def cell_edges(masses) -> np.ndarray:
    m = np.asarray(masses, dtype=np.float64)
    if m.ndim != 1 or m.size < 2 or np.any(np.diff(m) <= 0):
        raise ValueError("masses must be increasing")
    return np.concatenate([[m[0]], np.sqrt(m[:-1] * m[1:]), [m[-1]]])


def weights(masses, imf=KROUPA) -> np.ndarray:
    """imf_w of one isochrone: IMF integrated over each point's mass cell, normalised to sum 1."""
    c = cumulative(cell_edges(masses), imf)
    w = np.diff(c)
    return w / w.sum()
