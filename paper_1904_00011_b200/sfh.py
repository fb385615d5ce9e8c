"""Host-side parameter transforms of the paper's star-formation-history models S1-S5
(PAPER.md:141-151): free parameters -> stars per pixel per isochrone age, the `sfh[A]` array of
`pcmd_params`.  Argument preparation only: nothing here runs on the hot path, and the library takes
linear per-age star counts whatever produced them (DESIGN.md R-Q5).

Age grid: N_age bins equally spaced in log10(age/yr) between 6.0 and 10.2 (1 Myr to
~14 Gyr... the paper's mid-points 10^6.1, 10^6.3, ... 10^10.1 for N_age = 21), SFR constant inside a bin,
so a bin [a_lo, a_hi] (linear years) formed  integral of SFR(t) dt  stars.

Reading of the time variable of S3/S4 (the paper gives only "SFR ~ exp(-t/tau)" and "t exp(-t/tau)"): t
is the time since star formation began at the oldest edge of the grid, t = T_max - lookback age.
"""
from __future__ import annotations

import numpy as np

LOG_AGE_MIN, LOG_AGE_MAX = 6.0, 10.2


def age_edges(n_age: int = 21, lo: float = LOG_AGE_MIN, hi: float = LOG_AGE_MAX) -> np.ndarray:
    """log10 age edges of the N_age bins."""
    return np.linspace(lo, hi, n_age + 1)


def age_midpoints(n_age: int = 21) -> np.ndarray:
    e = age_edges(n_age)
    return 0.5 * (e[:-1] + e[1:])


def _normalise(w: np.ndarray, n_pix: float) -> np.ndarray:
    w = np.asarray(w, dtype=np.float64)
    return n_pix * w / w.sum()


def ssp(log_age: float, n_pix: float, n_age: int = 21) -> np.ndarray:
    """S1: all stars in the age bin that contains log_age."""
    e = age_edges(n_age)
    i = int(np.clip(np.searchsorted(e, log_age, side="right") - 1, 0, n_age - 1))
    out = np.zeros(n_age)
    out[i] = n_pix
    return out


def constant(n_pix: float, n_age: int = 21) -> np.ndarray:
    """S2: constant SFR: a bin's share is its width in linear time."""
    a = 10.0 ** age_edges(n_age)
    return _normalise(a[1:] - a[:-1], n_pix)


def tau_model(n_pix: float, tau_gyr: float, n_age: int = 21, delayed: bool = False) -> np.ndarray:
    """S3 (SFR ~ exp(-t/tau)) and S4 (delayed: SFR ~ t exp(-t/tau)), t = T_max - age, integrated
    exactly over every bin."""
    a = 10.0 ** age_edges(n_age)
    T, tau = a[-1], tau_gyr * 1e9
    t_hi, t_lo = T - a[:-1], T - a[1:]                 # a bin [a_lo, a_hi] is t in [T - a_hi, T - a_lo]
    x_lo, x_hi = t_lo / tau, t_hi / tau
    if not delayed:                                    # tau (e^-x_lo - e^-x_hi), written with expm1
        w = tau * (np.expm1(-x_lo) - np.expm1(-x_hi))
    else:                                              # integral of t e^(-t/tau) = tau^2 [h(x_hi) - h(x_lo)],
        h = lambda x: -np.expm1(-x) - x * np.exp(-x)   # h(x) = 1 - (1 + x) e^-x  (stable for small x)
        w = tau * tau * (h(x_hi) - h(x_lo))
    return _normalise(w, n_pix)


def non_parametric(log_sfh_bins, bin_edges, n_age: int = 21) -> np.ndarray:
    """S5: log10 stars per pixel formed in each coarse bin (edges in log10 age); SFR constant inside a
    coarse bin, so its stars are spread over the fine age bins in proportion to the linear-time
    overlap.  N_pix is the sum."""
    tot = 10.0 ** np.asarray(log_sfh_bins, dtype=np.float64)
    be = 10.0 ** np.asarray(bin_edges, dtype=np.float64)
    assert be.size == tot.size + 1 and np.all(np.diff(be) > 0)
    a = 10.0 ** age_edges(n_age)
    out = np.zeros(n_age)
    for k in range(tot.size):
        lo = np.maximum(a[:-1], be[k])
        hi = np.minimum(a[1:], be[k + 1])
        ov = np.clip(hi - lo, 0.0, None)
        if ov.sum() > 0:
            out += tot[k] * ov / (be[k + 1] - be[k])
    return out


def default_bins5() -> np.ndarray:
    """Five coarse bins aligned with the 21-bin grid (edges at log age 6.0, 8.0, 9.0, 9.6, 10.0, 10.2:
    the paper says only "by default: 5"; number and edges are hyper-parameters)."""
    return np.array([6.0, 8.0, 9.0, 9.6, 10.0, 10.2])
