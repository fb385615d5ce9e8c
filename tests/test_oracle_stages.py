"""Pins of the oracle's stages 1-7 against closed forms, invariants the paper states,
library routines (numpy.fft, numpy.histogram2d, scipy.stats) and brute force.  CPU only."""
import math
import os

import numpy as np
import pytest
from scipy import special, stats

from oracle import pcmd_oracle as O
from workloads import synthetic as W

GOLD = os.path.join(os.path.dirname(__file__), "golden")


@pytest.fixture(scope="module")
def c1():
    return W.config(1, allow_unfrozen=True)


@pytest.fixture(scope="module")
def c2small():
    return W.scaled(W.config(2, allow_unfrozen=True), 48)


# ------------------------------------------------------------------ stage 1
def test_stage1_sum_lambda_is_npix(c2small):
    # PAPER.md:71 "normalizing the weights to equal N_pix"
    o = O.Oracle(c2small)
    prm = c2small["params"][0]
    mdfw, lam, flux = o.stage1(prm)
    assert abs(lam.sum() - prm["sfh"].sum()) < 1e-12 * prm["sfh"].sum()
    assert abs(mdfw.sum() - 1) < 1e-14
    assert np.all(lam >= 0)


def test_stage1_mdf_golden_and_gaussian(c2small):
    o = O.Oracle(c2small)
    mdfw, _, _ = o.stage1(c2small["params"][0])
    with open(os.path.join(GOLD, "mdf_c2.txt")) as fh:
        want = [float(t) for ln in fh if not ln.startswith("#") for t in ln.split()]
    assert np.allclose(mdfw, want, atol=6e-5)
    g = stats.norm.pdf(c2small["feh_grid"], -0.5, 0.2)
    assert np.allclose(mdfw, g / g.sum(), rtol=1e-9)


def test_stage1_mdf_cut_and_offgrid(c2small):
    o = O.Oracle(c2small)
    prm = dict(c2small["params"][0])
    prm["feh_sigma"] = 0.05           # neighbours at e^-12.5 < 1 % -> removed
    mdfw, lam, _ = o.stage1(prm)
    assert list(mdfw) == [0, 0, 1, 0, 0]
    assert abs(lam.sum() - prm["sfh"].sum()) < 1e-9
    prm["feh_mean"] = 40.0            # far off the grid: degenerates to the nearest point, no 0/0
    mdfw, _, _ = o.stage1(prm)
    assert list(mdfw) == [0, 0, 0, 0, 1]
    prm["feh_mean"], prm["feh_sigma"] = -0.5, 0.45   # broad: three central points kept, edges > 1 % too
    mdfw, _, _ = o.stage1(prm)
    g = stats.norm.pdf(c2small["feh_grid"], -0.5, 0.45)
    assert np.allclose(mdfw, g / g.sum(), rtol=1e-9)


def test_stage1_one_hot_sfh_is_single_age(c2small):
    o = O.Oracle(c2small)
    prm = dict(c2small["params"][0])
    sfh = np.zeros(7)
    sfh[3] = 500.0
    prm["sfh"] = sfh
    _, lam, _ = o.stage1(prm)
    assert np.all(lam[c2small["age_idx"] != 3] == 0)
    assert abs(lam.sum() - 500.0) < 1e-10


def test_stage1_flux_zero_point_and_pogson(c1):
    o = O.Oracle(c1)
    prm = dict(c1["params"][0])
    _, _, f0 = o.stage1(prm)
    prm["dmod"] += 5.0                 # Pogson: 5 mag = factor 100 exactly
    _, _, f5 = o.stage1(prm)
    assert np.allclose(f0 / f5, 100.0, rtol=1e-12)
    # a star whose apparent magnitude equals the zero-point gives 1 electron
    wl = dict(c1)
    wl["absmag"] = np.full_like(c1["absmag"], c1["zp"][0] - 24.0)
    _, _, f = O.Oracle(wl).stage1(c1["params"][0])
    assert np.allclose(f, 1.0, rtol=1e-12)


# ------------------------------------------------------------------ stage 2
def test_stage2_closed_form_moments(c1):
    # compound Poisson: E F_b = sum lam f, Var F_b = sum lam f^2 ; total ~ Poisson(N_pix)
    o = O.Oracle(c1)
    _, lam, flux = o.stage1(c1["params"][0])
    F, total, _ = o.stage2(lam, flux, seed=0)
    P = o.P
    for b in range(o.B):
        mu, var = (lam * flux[:, b]).sum(), (lam * flux[:, b] ** 2).sum()
        m4 = (lam * flux[:, b] ** 4).sum() + 3 * var ** 2   # 4th central moment of compound Poisson
        assert abs(F[b].mean() - mu) < 5 * math.sqrt(var / P)
        assert abs(F[b].var() - var) < 5 * math.sqrt((m4 - var ** 2) / P)
    npix = lam.sum()
    assert abs(total.mean() - npix) < 5 * math.sqrt(npix / P)
    assert abs(total.var() - npix) < 5 * math.sqrt((npix + 2 * npix ** 2) / P)


def test_stage2_matches_brute_force_4x4():
    wl = W.tiny_model(n_im=4, J=9, B=2)
    o = O.Oracle(wl)
    _, lam, flux = o.stage1(wl["params"][0])
    F, total, h, counts = o.stage2(lam, flux, seed=42, model=3, want_counts=True)
    Fb, totb = o.stage2_brute(lam, flux, seed=42, model=3)
    assert np.array_equal(total, totb)
    assert np.allclose(F, Fb, rtol=1e-13)
    assert total.sum() > 100  # the case is not vacuous
    # per-point counts follow the stream map (R-C1) and the hash is sum n * (splitmix64(j)|1) mod 2^64
    tabs = [O.poisson_table(float(l)) for l in lam]
    for p in range(16):
        hh = 0
        for j in range(9):
            w = O.philox([42, 0], [p, j >> 2, 3, 0])
            n = O.poisson_draw(*tabs[j], int(w[j & 3]), linear=True)
            assert n == counts[p, j]
            hh = (hh + n * (O.splitmix64(j) | 1)) % 2 ** 64
        assert hh == int(h[p])
        assert counts[p].sum() == total[p]
        assert np.allclose(F[:, p], counts[p].astype(float) @ flux, rtol=1e-13)


def test_stage2_single_point_isochrone():
    wl = W.tiny_model(n_im=8, J=1, B=2)
    o = O.Oracle(wl)
    _, lam, flux = o.stage1(wl["params"][0])
    F, total, _ = o.stage2(lam, flux, seed=1)
    assert np.array_equal(F[0], total * flux[0, 0])
    assert np.array_equal(F[1], total * flux[0, 1])


def test_stage2_pixel_subset_equals_full(c1):
    o = O.Oracle(c1)
    _, lam, flux = o.stage1(c1["params"][0])
    F, total, h = o.stage2(lam, flux, seed=9, model=2)
    pix = np.array([0, 5, 63, 64, 4095, 1234], dtype=np.uint32)
    Fs, ts, hs = o.stage2(lam, flux, seed=9, model=2, pix=pix)
    assert np.array_equal(Fs, F[:, pix]) and np.array_equal(ts, total[pix]) and np.array_equal(hs, h[pix])
    # different seed / model give different realisations
    F2, _, _ = o.stage2(lam, flux, seed=10, model=2, pix=pix)
    F3, _, _ = o.stage2(lam, flux, seed=9, model=3, pix=pix)
    assert not np.array_equal(F2, Fs) and not np.array_equal(F3, Fs)


def test_npix_scaling_sbf_limit():
    # N_pix raises luminosity, lowers dispersion ~ N_pix^-1/2; collapses to the
    # integrated-light point
    wl = W.scaled(W.config(1, allow_unfrozen=True), 32)
    o = O.Oracle(wl)
    rel = []
    for npix in (1e2, 1e4, 1e6):
        prm = dict(wl["params"][0])
        prm["sfh"] = np.array([npix])
        _, lam, flux = o.stage1(prm)
        F, _, _ = o.stage2(lam, flux, seed=0)
        mu = (lam[:, None] * flux).sum(axis=0)
        sd = np.sqrt((lam[:, None] * flux ** 2).sum(axis=0))
        assert np.all(np.abs(F.mean(axis=1) / mu - 1) < 5 * sd / mu / math.sqrt(o.P))
        rel.append(F[1].std() / F[1].mean())
    assert 7 < rel[0] / rel[1] < 14 and 7 < rel[1] / rel[2] < 14
    mags = -2.5 * np.log10(F[1] / mu[1])
    assert np.abs(mags).max() < 6 * 1.0857 * sd[1] / mu[1]


# ------------------------------------------------------------------ stage 3
def _dusty(c1, mode, frac=0.5):
    wl = dict(c1)
    wl["dust_mode"], wl["dust_frac"] = mode, frac
    wl["dust_coef"] = np.array([1.2, 0.6])
    return wl


def test_stage3_limits(c1):
    F = np.random.default_rng(0).uniform(1, 2, size=(2, 4096))
    prm = dict(c1["params"][0], dust_med=0.5, dust_sigma=0.0)
    A, Fd = O.Oracle(_dusty(c1, 1, 1.0)).stage3(prm, F, seed=0)     # E1: constant screen
    assert np.allclose(A, 0.5)
    assert np.allclose(Fd[0] / F[0], 10 ** (-0.4 * 1.2 * 0.5), rtol=1e-14)
    assert np.allclose(Fd[1] / F[1], 10 ** (-0.4 * 0.6 * 0.5), rtol=1e-14)
    _, Fd = O.Oracle(_dusty(c1, 1, 0.0)).stage3(prm, F, seed=0)     # F_dust = 0: identity
    assert np.array_equal(Fd, F)
    _, Fd = O.Oracle(_dusty(c1, 0)).stage3(prm, F, seed=0)
    assert np.array_equal(Fd, F)
    _, Fd = O.Oracle(_dusty(c1, 1, 0.5)).stage3(prm, F, seed=0)     # mid-plane: half the stars reddened
    assert np.allclose(Fd[0] / F[0], 0.5 + 0.5 * 10 ** (-0.4 * 1.2 * 0.5), rtol=1e-14)


def test_stage3_lognormal_statistics(c1):
    F = np.ones((2, 4096))
    prm = dict(c1["params"][0], dust_med=0.5, dust_sigma=0.2)
    A, Fd = O.Oracle(_dusty(c1, 2, 0.3)).stage3(prm, F, seed=4)
    lnA = np.log(A)
    assert abs(np.median(A) - 0.5) < 0.5 * 0.2 * 5 * 1.2533 / math.sqrt(A.size)   # median = dust_med
    assert abs(lnA.std() - 0.2) < 5 * 0.2 / math.sqrt(2 * A.size)
    assert stats.kstest((lnA - math.log(0.5)) / 0.2, "norm").pvalue > 1e-3
    behind = Fd[0] != 1.0
    assert abs(behind.mean() - 0.3) < 5 * math.sqrt(0.21 / A.size)                # mode 2 fraction -> F_d
    assert np.allclose(Fd[0][behind], 10 ** (-0.4 * 1.2 * A[behind]), rtol=1e-13)
    assert np.allclose(np.log(Fd[0][behind]) / np.log(Fd[1][behind]), 2.0, rtol=1e-9)  # reddening law ratio


# ------------------------------------------------------------------ stage 4
def test_stage4_delta_identity_and_flux_conservation(c1):
    rng = np.random.default_rng(1)
    F = rng.gamma(2.0, 100.0, size=(2, 4096))
    wl = dict(c1)
    d = np.zeros((2, 5, 5))
    d[:, 2, 2] = 1
    wl["psf2d"] = d
    assert np.array_equal(O.Oracle(wl).stage4(F), F)
    G = O.Oracle(c1).stage4(F)
    assert np.allclose(G.sum(axis=1), F.sum(axis=1) * c1["psf2d"].sum(axis=(1, 2)), rtol=1e-12)


def test_stage4_equals_fft_circular_convolution():
    wl = W.with_psf(W.scaled(W.config(1, allow_unfrozen=True), 24), 7, [1.3, 0.9])
    rng = np.random.default_rng(2)
    # asymmetric kernel so that a flipped or transposed operand fails
    psf = rng.uniform(0, 1, size=(2, 7, 7))
    psf /= psf.sum(axis=(1, 2), keepdims=True)
    wl["psf2d"] = psf
    F = rng.gamma(2.0, 50.0, size=(2, 24 * 24))
    G = O.Oracle(wl).stage4(F)
    for b in range(2):
        k = np.zeros((24, 24))
        for dy in range(-3, 4):
            for dx in range(-3, 4):
                k[dy % 24, dx % 24] = psf[b, dy + 3, dx + 3]
        ref = np.real(np.fft.ifft2(np.fft.fft2(F[b].reshape(24, 24)) * np.fft.fft2(k)))
        assert np.allclose(G[b].reshape(24, 24), ref, rtol=1e-10, atol=1e-9)


def test_stage4_point_source_places_psf():
    wl = W.scaled(W.config(1, allow_unfrozen=True), 8)
    psf = np.arange(50, dtype=float).reshape(2, 5, 5) + 1
    wl["psf2d"] = psf
    F = np.zeros((2, 64))
    F[:, 1 * 8 + 7] = 1.0          # star at (y=1, x=7): wraps in x
    G = O.Oracle(wl).stage4(F).reshape(2, 8, 8)
    for dy in range(-2, 3):
        for dx in range(-2, 3):
            assert G[0, (1 + dy) % 8, (7 + dx) % 8] == psf[0, dy + 2, dx + 2]


# ------------------------------------------------------------------ stage 5
def test_stage5_noise_off_is_pogson(c1):
    wl = dict(c1)
    wl["shot_noise"], wl["read_sigma"] = 0, np.zeros(2)
    G = np.stack([np.full(4096, 1.0), np.full(4096, 100.0)])
    mag = O.Oracle(wl).stage5(G, seed=0)
    assert np.allclose(mag[0], c1["zp"][0], atol=1e-13)
    assert np.allclose(mag[1], c1["zp"][1] - 5.0, atol=1e-13)
    G[0, 0] = 0.0
    G[0, 1] = -3.0
    mag = O.Oracle(wl).stage5(G, seed=0)
    assert np.isnan(mag[0, 0]) and np.isnan(mag[0, 1]) and not np.isnan(mag[0, 2])


def test_stage5_noise_statistics(c1):
    P = 4096
    wl = dict(c1)
    wl["shot_noise"], wl["read_sigma"], wl["sky"], wl["poisson_sky"] = 1, np.array([5.0, 0.0]), np.array([50.0, 0.0]), 0
    G = np.stack([np.full(P, 400.0), np.full(P, 900.0)])
    mag = O.Oracle(wl).stage5(G, seed=3)
    C = 10 ** (-0.4 * (mag - c1["zp"][:, None]))           # = C' - sky
    for b, (mu, var) in enumerate([(400.0, 450.0 + 25.0), (900.0, 900.0)]):   # noise = sqrt(counts)
        assert abs(C[b].mean() - mu) < 5 * math.sqrt(var / P)
        assert abs(C[b].var() - var) < 5 * var * math.sqrt(2.0 / P)
        assert stats.kstest((C[b] - mu) / math.sqrt(var), "norm").pvalue > 1e-3
    # Poisson sky: integer sky counts with mean = var = sky, on top of Gaussian shot+read noise
    wl["poisson_sky"], wl["shot_noise"], wl["read_sigma"] = 1, 0, np.zeros(2)
    mag = O.Oracle(wl).stage5(G, seed=3)
    K = 10 ** (-0.4 * (mag[0] - c1["zp"][0])) - 400.0 + 50.0
    assert np.allclose(K, np.round(K), atol=1e-8)
    assert abs(K.mean() - 50) < 5 * math.sqrt(50 / P) and abs(K.var() - 50) < 5 * 50 * math.sqrt(2.2 / P)


def test_distance_modulus_only_shifts_magnitudes():
    # PAPER.md:186 "simply shifts the distribution in the vertical (luminosity) direction, with no effect on color"
    wl = W.scaled(W.config(1, allow_unfrozen=True), 16)
    wl["shot_noise"], wl["read_sigma"] = 0, np.zeros(2)
    o = O.Oracle(wl)
    a = o.simulate(wl["params"][0], seed=0)
    prm = dict(wl["params"][0])
    prm["dmod"] += 1.25
    b = o.simulate(prm, seed=0)
    assert np.array_equal(a["total"], b["total"])           # counts do not depend on distance (R-Q1)
    assert np.allclose(b["mag"] - a["mag"], 1.25, atol=1e-11)


# ------------------------------------------------------------------ stage 6
def _hspec(nx=20, ny=30):
    return dict(band_plus=0, band_minus=1, band_y=1, x_lo=-1.0, x_hi=3.0, y_lo=18.0, y_hi=30.0, nx=nx, ny=ny)


def test_hess_equals_numpy_histogram2d(c1):
    rng = np.random.default_rng(8)
    P = 20000
    m1 = rng.uniform(17, 31, P)
    m0 = m1 + rng.normal(1.0, 1.2, P)
    m0[::97] = np.nan
    mag = np.stack([m0, m1])
    h = _hspec()
    H, st = O.Oracle(c1).hess(h, mag)
    ok = ~np.isnan(m0)
    x, y = (m0 - m1)[ok], m1[ok]
    ref, _, _ = np.histogram2d(y, x, bins=[h["ny"], h["nx"]], range=[[18, 30], [-1, 3]])
    # numpy closes the last bin on the right; ours is half-open -- no sample sits exactly on an edge here
    assert np.array_equal(H, ref.astype(np.uint32))
    assert st["n_bad"] == (~ok).sum()
    assert st["n_in"] + st["n_out"] + st["n_bad"] == P and st["n_in"] == H.sum()
    inw = (x >= -1) & (x < 3) & (y >= 18) & (y < 30)
    assert abs(st["sum_x"] - x[inw].sum()) < 1e-8 and abs(st["sum_y"] - y[inw].sum()) < 1e-7


def test_hess_half_open_edges_and_edge_count(c1):
    h = _hspec(nx=4, ny=12)     # dx = 1, dy = 1
    # points: exactly on lower edge (in bin 0), on upper edge (out), on an inner edge (upper bin), near an edge
    x = np.array([-1.0, 3.0, 1.0, 0.5, 0.5 + 0.5 - 4e-6, 0.5])
    y = np.array([18.5, 18.5, 18.5, 30.0, 20.5, 18.0])
    mag = np.stack([x + y, y])
    H, st = O.Oracle(c1).hess(h, mag, edge_tol=1e-5, want_edges=True)
    assert H[0, 0] == 1 and H[0, 2] == 1 and H[2, 1] == 1 and H[0, 1] == 1
    assert st["n_out"] == 2 and st["n_in"] == 4
    assert st["n_edge"] == 6 and list(st["edges"]) == [0, 1, 2, 3, 4, 5]
    mag2 = np.stack([np.array([0.5 + 19.3]), np.array([19.3])])
    _, st2 = O.Oracle(c1).hess(h, mag2)
    assert st2["n_edge"] == 0


def test_hess_f32_agrees_with_f64_away_from_edges(c1):
    rng = np.random.default_rng(9)
    P = 50000
    m1 = rng.uniform(17, 31, P).astype(np.float32)
    m0 = (m1 + rng.normal(1.0, 1.2, P)).astype(np.float32)
    mag32 = np.stack([m0, m1])
    h = _hspec(64, 64)
    o = O.Oracle(c1)
    H32, s32 = o.hess_f32(h, mag32)
    H64, s64 = o.hess(h, mag32.astype(np.float64), edge_tol=1e-5)
    assert np.abs(H32.astype(int) - H64.astype(int)).sum() <= 2 * s64["n_edge"]
    assert s32["n_in"] + s32["n_out"] + s32["n_bad"] == P


def test_hess_pixels_is_the_per_pixel_form_of_hess(c1):
    """orc_hess_pixels / orc_hess_pixels_f32 (used by the GPU parity tests for the per-pixel edge-membership
    check) against orc_hess / orc_hess_f32 and against plain numpy floor arithmetic."""
    rng = np.random.default_rng(12)
    P = 30000
    m1 = rng.uniform(17, 31, P)
    m0 = m1 + rng.normal(1.0, 1.2, P)
    m0[::101] = np.nan
    # a few pixels a hair away from an edge on either axis
    m1[5], m0[5] = 20.0 + 6e-6, 20.0 + 6e-6 + 0.55
    m1[6], m0[6] = 22.3, 22.3 + 1.0 - 1.5e-5          # x within 2e-5, not within 1e-5
    mag = np.stack([m0, m1])
    h = _hspec(40, 60)     # dx = 0.1, dy = 0.2
    o = O.Oracle(c1)
    H, st = o.hess(h, mag, edge_tol=1e-5, want_edges=True)
    b, near = o.hess_pixels(h, mag, tol_x=1e-5, tol_y=1e-5)
    assert np.array_equal(np.bincount(b[b >= 0], minlength=h["nx"] * h["ny"]).reshape(h["ny"], h["nx"]), H)
    assert (b == -2).sum() == st["n_bad"] and (b == -1).sum() == st["n_out"]
    assert np.array_equal(np.nonzero(near)[0].astype(np.uint32), st["edges"])
    assert near[5] == 2 and near[6] == 0
    _, near2 = o.hess_pixels(h, mag, tol_x=2e-5, tol_y=1e-5)
    assert near2[6] == 1 and np.all((near2 & 2) == (near & 2)) and np.all(near2 >= near)
    # plain numpy definition of the bin index
    ok = ~np.isnan(m0)
    ix = np.floor(((m0 - m1) - h["x_lo"]) / ((h["x_hi"] - h["x_lo"]) / h["nx"]))
    iy = np.floor((m1 - h["y_lo"]) / ((h["y_hi"] - h["y_lo"]) / h["ny"]))
    inw = ok & (ix >= 0) & (ix < h["nx"]) & (iy >= 0) & (iy < h["ny"])
    assert np.array_equal(b[inw], (iy[inw] * h["nx"] + ix[inw]).astype(np.int32))
    assert np.all(b[ok & ~inw] == -1)
    # fp32 form
    mag32 = mag.astype(np.float32)
    H32, s32 = o.hess_f32(h, mag32)
    b32 = o.hess_pixels_f32(h, mag32)
    assert np.array_equal(np.bincount(b32[b32 >= 0], minlength=h["nx"] * h["ny"]).reshape(h["ny"], h["nx"]), H32)
    assert (b32 == -2).sum() == s32["n_bad"] and (b32 == -1).sum() == s32["n_out"]
    # away from edges both precisions agree pixel by pixel
    b64, near64 = o.hess_pixels(h, mag32.astype(np.float64), tol_x=2e-5, tol_y=1e-5)
    assert np.all((b32 == b64) | (near64 != 0))


# ------------------------------------------------------------------ stage 7
def test_loglike_poisson_vs_scipy():
    rng = np.random.default_rng(10)
    m = rng.poisson(3.0, size=400).astype(np.uint32)
    d = rng.poisson(3.0, size=400).astype(np.uint32)
    m[:50] = 0
    d[25:75] = 0
    s = d.sum() / m.sum()
    mu = s * np.maximum(m.astype(float), 0.1)
    use = (d > 0) | (m > 0)
    ref = stats.poisson.logpmf(d[use], mu[use]).sum()
    assert abs(O.loglike_poisson(m, d, 0.1) - ref) < 1e-9 * abs(ref)
    # model == data: sum d ln d - d - lgamma(d+1)
    dd = d[d > 0].astype(float)
    ref2 = (dd * np.log(dd) - dd - special.gammaln(dd + 1)).sum()
    assert abs(O.loglike_poisson(d, d, 0.1) - ref2) < 1e-9 * abs(ref2)
    # a data pixel in an empty model bin costs a finite amount (the floor), not -inf
    m2, d2 = np.array([10, 0], dtype=np.uint32), np.array([9, 1], dtype=np.uint32)
    assert np.isfinite(O.loglike_poisson(m2, d2, 0.1))
    assert O.loglike_poisson(m2, d2, 0.1) < O.loglike_poisson(np.array([9, 1], dtype=np.uint32), d2, 0.1)


def test_loglike_gauss_eq2_to_4():
    rng = np.random.default_rng(12)
    d = rng.poisson(5.0, size=100).astype(np.uint32)
    sd = dict(n_in=int(d.sum()), n_out=0, n_bad=0, sum_x=0.7 * d.sum(), sum_y=24.0 * d.sum())
    # identical Hess: Eq. 2 sum = 0 and Eq. 4 = 0
    assert O.loglike_gauss(d, sd, d, sd) == 0.0
    assert O.loglike_gauss(d, sd, d, sd, literal=True) == 0.0
    # Eq. 4 alone: same Hess, mean colour offset by 0.05 mag -> -1/2
    sm = dict(sd, sum_x=(0.7 + 0.05) * d.sum())
    assert abs(O.loglike_gauss(d, sm, d, sd) + 0.5) < 1e-9
    # equal totals: sigma^2 = (max(d,1) + max(m,1))/N^2 >= 2/N^2 -- the printed floor "2" (R-Q14)
    m = np.roll(d, 1)
    N = float(d.sum())
    ref = -(((d / N - m / N) ** 2) / (2 * (np.maximum(d, 1) + np.maximum(m, 1)) / N ** 2)).sum()
    assert abs(O.loglike_gauss(m, sd, d, sd) - ref) < 1e-12 * abs(ref)
    lit = -(((d / N - m / N) ** 2) / (2 * np.maximum(np.sqrt(d.astype(float) ** 2 + m.astype(float) ** 2), 2) ** 2)).sum()
    assert abs(O.loglike_gauss(m, sd, d, sd, literal=True) - lit) < 1e-12 * abs(lit)


def test_loglike_is_stochastic_and_tightens_with_nim():
    # a new realisation every call; scatter decreases with N_im
    base = W.config(1, allow_unfrozen=True)
    sc = []
    for n in (16, 48):
        wl = W.scaled(base, n)
        o = O.Oracle(wl)
        h = wl["hess"][0]
        Hd, _ = o.hess(h, o.simulate(wl["params"][0], seed=100)["mag"])
        ll = []
        for s in range(8):
            Hm, _ = o.hess(h, o.simulate(wl["params"][0], seed=s)["mag"])
            ll.append(O.loglike_poisson(Hm, Hd) / Hd.sum())
        sc.append(np.std(ll))
        assert len(set(ll)) == 8
    assert sc[1] < sc[0]


# ---- sub-pixel PSF grid (DESIGN.md R-Q19) ------------------------------------------
def test_psf_grid_with_identical_psfs_equals_the_single_psf():
    wl = W.scaled(W.config(2), 20)
    G = 4
    g = dict(wl, psf_grid=G, psf_grid2d=np.repeat(wl["psf2d"][:, None], G * G, axis=1))
    rng = np.random.default_rng(5)
    F = rng.uniform(1.0, 100.0, size=(wl["n_bands"], 400))
    assert np.array_equal(O.Oracle(g).stage4(F), O.Oracle(wl).stage4(F))


def test_psf_grid_of_shifted_deltas_shifts_every_cell_by_its_own_offset():
    """Each cell's PSF is a delta at a different whole-pixel offset: the output pixel (y, x) of cell c
    must be the input pixel (y - dy_c, x - dx_c) (circular) -- brute force with numpy indexing."""
    wl = W.scaled(W.config(2), 10)          # cells of ceil(10/4) = 3 pixels: 3,3,3,1
    K, B, G, N = int(wl["psf_k"]), int(wl["n_bands"]), 4, 10
    r = (K - 1) // 2
    rng = np.random.default_rng(6)
    offs = rng.integers(-r, r + 1, size=(B, G * G, 2))
    psf = np.zeros((B, G * G, K, K), dtype=np.float32)
    for b in range(B):
        for c in range(G * G):
            psf[b, c, offs[b, c, 0] + r, offs[b, c, 1] + r] = 1.0
    F = rng.uniform(1.0, 100.0, size=(B, N * N))
    got = O.Oracle(dict(wl, psf_grid=G, psf_grid2d=psf)).stage4(F).reshape(B, N, N)
    cell = -(-N // G)
    for b in range(B):
        Fb = F[b].reshape(N, N)
        for y in range(N):
            for x in range(N):
                c = min(G - 1, y // cell) * G + min(G - 1, x // cell)
                dy, dx = offs[b, c]
                assert got[b, y, x] == Fb[(y - dy) % N, (x - dx) % N]


def test_psf_grid_generator_is_normalised_and_shifted():
    wl = W.with_psf_grid(W.scaled(W.config(3), 16), 4)
    p = wl["psf_grid2d"].astype(np.float64)
    assert p.shape == (3, 16, 15, 15)
    assert np.allclose(p.sum(axis=(2, 3)), 1.0, atol=1e-6)
    d = np.arange(-7, 8)
    cx = (p * d[None, None, None, :]).sum(axis=(2, 3))           # centroid in x per (band, cell)
    want = (np.arange(4) + 0.5) / 4 - 0.5
    assert np.allclose(cx[0].reshape(4, 4)[0], want, atol=2e-3)
