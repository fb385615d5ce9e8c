"""Host-side transform of the paper's dust parameter: E(B-V) -> per-band extinction A_b
("the dust extinction in units of the reddening parameter log E(B-V)", an R_V = 3.1
reddening law).  Argument preparation only: the library takes `dust_coef[b]` = A_b per unit of the dust
parameter (pcmd_config) and the per-pixel dust parameter is drawn around `dust_med` (pcmd_params), so
with dust_med = E(B-V) the coefficients are A_b / E(B-V) = R_V * A_b / A_V.

The filter response curves the paper integrates over (ACS filters) are not available here;
the law is evaluated at a band's effective wavelength.  The curve is the mean R_V-dependent extinction
law of Cardelli, Clayton & Mathis (1989) in its infrared and optical/near-infrared ranges,
A(x)/A_V = a(x) + b(x)/R_V with x = 1/lambda in inverse microns, restated from the published
polynomial.
"""
from __future__ import annotations

import numpy as np

R_V_DEFAULT = 3.1


def extinction_ratio(wavelength_um, r_v: float = R_V_DEFAULT) -> np.ndarray:
    """A(lambda)/A_V for 0.3 <= 1/lambda <= 3.3 per micron (0.303 ... 3.33 micron)."""
    x = 1.0 / np.atleast_1d(np.asarray(wavelength_um, dtype=np.float64))
    if np.any(x < 0.3) or np.any(x > 3.3):
        raise ValueError("wavelength outside the infrared / optical range of the law (0.303-3.33 micron)")
    a = np.empty_like(x)
    b = np.empty_like(x)
    ir = x < 1.1
    a[ir] = 0.574 * x[ir] ** 1.61
    b[ir] = -0.527 * x[ir] ** 1.61
    y = x[~ir] - 1.82
    # Horner form of the two degree-7 polynomials in y = x - 1.82
    ca = (1.0, 0.17699, -0.50447, -0.02427, 0.72085, 0.01979, -0.77530, 0.32999)
    cb = (0.0, 1.41338, 2.28305, 1.07233, -5.38434, -0.62251, 5.30260, -2.09002)
    pa = np.zeros_like(y)
    pb = np.zeros_like(y)
    for c_a, c_b in zip(reversed(ca), reversed(cb)):
        pa = pa * y + c_a
        pb = pb * y + c_b
    a[~ir] = pa
    b[~ir] = pb
    return a + b / r_v


def dust_coef_per_ebv(wavelength_um, r_v: float = R_V_DEFAULT) -> np.ndarray:
    """`dust_coef[b]` for a dust parameter in units of E(B-V): A_b / E(B-V) = R_V * A(lambda_b)/A_V."""
    return r_v * extinction_ratio(wavelength_um, r_v)


def dust_coef_per_av(wavelength_um, r_v: float = R_V_DEFAULT) -> np.ndarray:
    """`dust_coef[b]` for a dust parameter in units of A_V (BASELINE.json's c3: "log-normal A_V")."""
    return extinction_ratio(wavelength_um, r_v)
