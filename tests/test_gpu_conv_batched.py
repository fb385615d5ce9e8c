"""Stages 4-5 on GPU-filling batches: the register-blocked separable kernel k_conv2 (taken when one launch per
band fills the GPU, csrc/conv_noise.cu) against the oracle's quadruple-loop convolution and its stage 5, for
every compiled PSF size, image sizes that are / are not multiples of the tile and of four, with the noise of
c1 (read noise) and of c3 (Poisson sky + shot + read noise).  PAPER.md:83,127-128,178; R-Q9, R-Q11."""
import numpy as np
import pytest

from oracle import pcmd_oracle as O
from workloads import synthetic as W
from _parity import FLUX_RTOL, MAG_ATOL

pytestmark = pytest.mark.gpu


@pytest.mark.parametrize("cfg,K,sig,n_im,n_models", [
    (1, 5, 1.0, 64, 300), (1, 7, 1.0, 66, 80), (1, 15, 1.5, 128, 80), (1, 21, 2.0, 72, 80),
    (3, 15, 1.2, 64, 300), (3, 7, 1.0, 33, 300)])
def test_batched_separable_convolution_and_noise(cfg, K, sig, n_im, n_models):
    import torch
    import paper_1904_00011_b200 as G
    base = W.config(cfg)
    wl = W.with_psf(W.scaled(base, n_im), K, [sig] * int(base["n_bands"]))
    prm = [dict(wl["params"][0], dmod=wl["params"][0]["dmod"] + 0.01 * (i % 7)) for i in range(n_models)]
    if cfg == 3:                      # c3's tables and noise model with few stars per pixel: stage 2 is not under test here
        prm = [dict(p, sfh=np.asarray(p["sfh"]) * 0.02) for p in prm]
    g = G.Pcmd(wl, separable=True)
    P = g.N * g.N
    fd = torch.empty((n_models, g.B, g.N, g.N), dtype=torch.float32, device="cuda")
    fc = torch.empty_like(fd)
    g.debug_taps(fd, fc)
    seed, m0 = 23, 5
    out = g.simulate(prm, seed=seed, model_index0=m0)
    torch.cuda.synchronize()
    assert g.status() == 0
    orc = O.Oracle(wl)
    for i in (0, n_models // 2, n_models - 1):
        F = fd[i].cpu().numpy().reshape(g.B, P).astype(np.float64)
        Gc = orc.stage4(F)
        got = fc[i].cpu().numpy().reshape(g.B, P)
        scale = np.abs(Gc).max(axis=1, keepdims=True)
        assert np.max(np.abs(got - Gc) / np.maximum(np.abs(Gc), 1e-6 * scale)) <= FLUX_RTOL
        want = orc.stage5(got.astype(np.float64), seed, model=m0 + i)      # stage 5 isolated: the GPU's own convolved flux
        mag = out["mag"][i].cpu().numpy().reshape(g.B, P)
        ok = ~np.isnan(want)
        assert np.array_equal(np.isnan(mag), ~ok)
        assert np.max(np.abs(mag[ok] - want[ok])) <= MAG_ATOL
    g.debug_taps(None, None)
    g.close()


@pytest.mark.parametrize("read_sigma", [0.0, 3.0])
def test_batched_magnitude_of_non_positive_flux_is_nan(read_sigma):
    """Stage 5 on k_conv2 for fluxes <= 0 (R-Q11: the magnitude of a non-positive flux is NaN): a model without stars
    (every flux exactly 0: lg2 = -inf, the kernel's NaN comes out of (+inf) + (-inf), csrc/conv_noise.cu mag_of) and, with
    read noise and no sky, a sparse model whose noisy fluxes are negative in about half of the empty pixels."""
    import torch
    import paper_1904_00011_b200 as G
    base = W.config(1)
    wl = dict(W.with_psf(W.scaled(base, 64), 7, [1.0] * int(base["n_bands"])))
    wl["sky"] = np.zeros_like(wl["sky"])
    wl["read_sigma"] = np.full_like(wl["read_sigma"], read_sigma)
    wl["shot_noise"], wl["poisson_sky"] = 0, 0
    n_models = 300
    p0 = wl["params"][0]
    prm = [dict(p0, sfh=np.asarray(p0["sfh"]) * (0.0 if i % 2 == 0 else 1e-4)) for i in range(n_models)]
    g = G.Pcmd(wl, separable=True)
    P = g.N * g.N
    fc = torch.empty((n_models, g.B, g.N, g.N), dtype=torch.float32, device="cuda")
    g.debug_taps(None, fc)
    seed, m0 = 31, 2
    out = g.simulate(prm, seed=seed, model_index0=m0)
    torch.cuda.synchronize()
    assert g.status() == 0
    orc = O.Oracle(wl)
    n_nan = 0
    for i in (0, 1, n_models - 2, n_models - 1):
        got = fc[i].cpu().numpy().reshape(g.B, P)
        if i % 2 == 0:
            assert not got.any()                                            # no stars: flux exactly zero everywhere
        want = orc.stage5(got.astype(np.float64), seed, model=m0 + i)
        mag = out["mag"][i].cpu().numpy().reshape(g.B, P)
        ok = ~np.isnan(want)
        assert np.array_equal(np.isnan(mag), ~ok)
        assert not np.isinf(mag).any()
        if ok.any():
            # a flux that is the noise draw alone (|flux| << sigma) is ill-conditioned in magnitudes (d mag = 1.09 d flux /
            # flux, d flux = sigma x the fp32 error of the normal draw): compare it as a flux, on the scale of sigma
            zp = np.asarray(wl["zp"], dtype=np.float64)[:, None]
            f_got, f_want = 10.0 ** (-0.4 * (mag - zp)), 10.0 ** (-0.4 * (want - zp))
            assert np.max(np.abs(f_got[ok] - f_want[ok]) - FLUX_RTOL * np.abs(f_want[ok])) <= 1e-5 * max(read_sigma, 1e-30)
            well = ok & (f_want > max(read_sigma, 1e-30))
            if well.any():
                assert np.max(np.abs(mag[well] - want[well])) <= MAG_ATOL
        n_nan += int((~ok).sum())
        if read_sigma == 0.0 and i % 2 == 0:
            assert not ok.any()
    assert n_nan > P                                                        # the case is exercised
    g.debug_taps(None, None)
    g.close()
