"""Parity at BASELINE.json's full sizes, in the launch configuration bench.py times (separable PSF,
production kernels).  Stage 2 (the Monte Carlo part): sampled pixels, which the oracle computes one
by one -- counts bit-exact, flux 1e-5.  Stages 3-5: the oracle run on the GPU's own raw flux
(stage-isolated, every pixel).  Stage 6: exact in the kernel's precision; counts add up."""
import numpy as np
import pytest

from oracle import pcmd_oracle as O
from workloads import synthetic as W

pytestmark = pytest.mark.gpu


@pytest.mark.parametrize("c,models", [(2, [0]), (3, [0]), (4, [0, 17, 63]), (5, [0])])
def test_full_size_config(c, models):
    import torch
    import paper_1904_00011_b200 as G
    wl = W.config(c)
    seed = int(wl["seed"])
    g = G.Pcmd(wl, separable=True)
    prms = wl["params"]
    out = g.simulate(prms, seed=seed, want_raw=True, want_counts=True)
    fast = g.simulate(prms, seed=seed, want_raw=True)                  # production kernel
    H, st = g.hess(fast["mag"])
    torch.cuda.synchronize()
    assert g.status() == 0
    assert torch.equal(out["flux_raw"], fast["flux_raw"])
    orc = O.Oracle(wl)
    rng = np.random.default_rng(1234 + c)
    pix = np.unique(np.concatenate([rng.integers(0, g.P, 1500), [0, g.N - 1, g.P - g.N, g.P - 1]])).astype(np.uint32)
    stn = G.Pcmd.stats_to_numpy(st)
    for m in models:
        mdfw, lam, flux = orc.stage1(prms[m])
        w = g.debug_weights(m)
        assert np.array_equal(w["lam"], lam)
        F, tot, hsh = orc.stage2(lam, flux, seed, model=m, pix=pix)
        assert np.array_equal(out["total"][m].cpu().numpy().view(np.uint32)[pix], tot)
        assert np.array_equal(out["hash"][m].cpu().numpy().view(np.uint64)[pix], hsh)
        raw = fast["flux_raw"][m].cpu().numpy().reshape(g.B, -1)
        assert np.allclose(raw[:, pix], F, rtol=1e-5, atol=0)
        # stages 3-5 on the GPU's raw flux
        _, Fd = orc.stage3(prms[m], raw.astype(np.float64), seed, model=m)
        mag_o = orc.stage5(orc.stage4(Fd), seed, model=m)
        mag = fast["mag"][m].cpu().numpy().reshape(g.B, -1)
        ok = ~np.isnan(mag_o)
        assert np.array_equal(np.isnan(mag), ~ok)
        assert np.max(np.abs(mag[ok] - mag_o[ok])) <= 1e-5
        off = 0
        for hi, h in enumerate(wl["hess"]):
            nb = h["nx"] * h["ny"]
            Hg = H[m].cpu().numpy().view(np.uint32)[off:off + nb].reshape(h["ny"], h["nx"])
            off += nb
            H32, s32 = orc.hess_f32(h, mag)
            assert np.array_equal(Hg, H32)
            assert int(Hg.sum()) + int(stn[m, hi]["n_out"]) + int(stn[m, hi]["n_bad"]) == g.P
    g.close()


@pytest.mark.parametrize("c", [2, 3, 5])
def test_full_size_closed_forms(c):
    """Properties that hold at any size (north_star): over the pixels of a full-size image the raw flux
    has mean sum(lambda f) and variance sum(lambda f^2) (compound Poisson), and the star count per pixel
    is Poisson(N_pix): mean = variance = N_pix (footnote 3).  lambda and f from the ORACLE."""
    import torch
    import paper_1904_00011_b200 as G
    wl = W.config(c)
    g = G.Pcmd(wl, separable=True)
    prm = wl["params"][0]
    out = g.simulate([prm], seed=11, want_raw=True, want_counts=True)
    torch.cuda.synchronize()
    assert g.status() == 0
    _, lam, flux = O.Oracle(wl).stage1(prm)
    F = out["flux_raw"][0].cpu().numpy().reshape(g.B, -1).astype(np.float64)
    tot = out["total"][0].cpu().numpy().view(np.uint32).astype(np.float64)
    P = g.P
    n_pix = lam.sum()
    assert abs(tot.mean() - n_pix) <= 5 * np.sqrt(n_pix / P)
    assert abs(tot.var() - n_pix) <= 5 * n_pix * np.sqrt(2.0 / P) + 5 * np.sqrt(n_pix / P)
    for b in range(g.B):
        m1, m2 = (lam * flux[:, b]).sum(), (lam * flux[:, b] ** 2).sum()
        m4 = (lam * flux[:, b] ** 4).sum()
        assert abs(F[b].mean() - m1) <= 5 * np.sqrt(m2 / P)
        # variance of the sample variance of a compound Poisson sum: (kappa_4 + 2 sigma^4) / P, kappa_4 = sum(lambda f^4)
        assert abs(F[b].var() - m2) <= 5 * np.sqrt((m4 + 2 * m2 * m2) / P)
    g.close()
