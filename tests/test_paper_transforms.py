"""Host-side transforms of the paper's free parameters (PAPER.md:99-119 Table 1, :157 IMF, :159-165 dust):
pcmd_params_from_paper (C library, host only), the R_V reddening law, the IMF weights."""
import ctypes as C

import numpy as np
import pytest

from paper_1904_00011_b200 import binding, dust, imf


def test_params_from_paper_maps_log_parameters_to_linear_fields():
    ls = np.array([-np.inf, 0.0, 1.5, 2.0])
    p = binding.params_from_paper(ls, feh=-0.5, sigma_feh=0.2, log10_ebv=-0.5, sigma_dust=0.3, dmod=27.5)
    assert np.array_equal(p["sfh"], [0.0, 1.0, 10.0 ** 1.5, 100.0])
    assert p["feh_mean"] == -0.5 and p["feh_sigma"] == 0.2 and p["dmod"] == 27.5 and p["dust_sigma"] == 0.3
    assert p["dust_med"] == 10.0 ** -0.5
    assert abs(p["sfh"].sum() - (1 + 10 ** 1.5 + 100)) < 1e-12          # N_pix = sum of the SFH


@pytest.mark.parametrize("bad", [dict(sigma_feh=0.0), dict(sigma_dust=-1.0), dict(dmod=np.nan), dict(feh=np.inf)])
def test_params_from_paper_rejects_bad_input(bad):
    kw = dict(feh=-0.5, sigma_feh=0.2, log10_ebv=-0.5, sigma_dust=0.3, dmod=27.5)
    kw.update(bad)
    with pytest.raises(binding.PcmdError):
        binding.params_from_paper(np.zeros(3), **kw)
    L = binding.lib()
    assert L.pcmd_params_from_paper(3, None, -0.5, 0.2, -0.5, 0.3, 27.5, None, None) == -1


def test_reddening_law_fixed_points():
    # V band (x = 1.82 per micron): A/A_V = 1 by construction; E(B-V) = A_B - A_V = A_V / R_V within a few per cent
    assert abs(dust.extinction_ratio(1.0 / 1.82)[0] - 1.0) < 1e-12
    for rv in (3.1, 5.0):
        ab, av = dust.extinction_ratio([0.44, 0.55], rv)
        assert abs(rv * (ab - av) - 1.0) < 0.04
    # the two published branches meet at x = 1.1 per micron, the curve rises towards the blue, I band ~ 0.6 A_V
    lo, hi = dust.extinction_ratio([1.0 / 1.0999, 1.0 / 1.1001])
    assert abs(lo - hi) < 5e-3
    w = np.linspace(0.32, 3.0, 200)
    assert np.all(np.diff(dust.extinction_ratio(w)) < 0)
    assert 0.55 < dust.extinction_ratio(0.80)[0] < 0.65
    assert np.allclose(dust.dust_coef_per_ebv([0.55]), 3.1 * dust.extinction_ratio([0.55]))
    with pytest.raises(ValueError):
        dust.extinction_ratio(0.1)


def test_imf_weights_closed_forms():
    m = np.geomspace(0.1, 50.0, 300)
    w = imf.weights(m, imf.SALPETER)
    e = imf.cell_edges(m)
    want = e[:-1] ** -1.35 - e[1:] ** -1.35
    assert np.allclose(w, want / want.sum(), rtol=1e-12) and abs(w.sum() - 1.0) < 1e-12
    # Kroupa: continuous at the breaks, slopes -0.3 / -1.3 / -2.3 ("Kroupa & Pavel 2001")
    d = 1e-6
    for brk in (0.08, 0.5):
        left = np.diff(imf.cumulative([brk - d, brk]))[0] / d
        right = np.diff(imf.cumulative([brk, brk + d]))[0] / d
        assert abs(left / right - 1.0) < 1e-4
    for lo, hi, alpha in ((0.02, 0.07, 0.3), (0.1, 0.4, 1.3), (0.6, 30.0, 2.3)):
        num = np.diff(imf.cumulative([lo, lo * (1 + d)]))[0] / (lo * d)
        den = np.diff(imf.cumulative([hi, hi * (1 + d)]))[0] / (hi * d)
        assert abs(np.log(num / den) / np.log(hi / lo) - alpha) < 1e-3
    wk = imf.weights(m, imf.KROUPA)
    assert abs(wk.sum() - 1.0) < 1e-12 and np.all(wk > 0)
    # fewer low-mass stars per high-mass star than Salpeter
    assert wk[m < 0.3].sum() / wk[m > 1].sum() < w[m < 0.3].sum() / w[m > 1].sum()
