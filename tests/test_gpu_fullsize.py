"""Parity at BASELINE.json's full sizes, in the launch configuration bench.py times (separable PSF,
production kernels), against the fp64 oracle run on the WHOLE image end to end: every pixel of every
stage, the Hess per-pixel edge rule and the log-likelihood (tests/_parity.py states the rules)."""
import numpy as np
import pytest

from oracle import pcmd_oracle as O
from workloads import synthetic as W
from _parity import EDGE_TOL_X, EDGE_TOL_Y, FLUX_RTOL, MAG_ATOL, hess_pixel_parity, lnl_poisson_parity

pytestmark = pytest.mark.gpu


@pytest.mark.parametrize("c,models", [(2, [0]), (3, [0]), (4, [0, 17, 63]), (5, [0])])
def test_full_size_config(c, models):
    """Whole image, every pixel, against the fp64 oracle run end to end (PAPER.md:71,81,83 stages 1-5, :218
    stage 6, north_star stage 7): counts bit-exact, raw / dusty / convolved flux 1e-5 relative, magnitudes
    1e-5 mag, Hess per-pixel edge-membership rule, lnL 1e-4."""
    import torch
    import paper_1904_00011_b200 as G
    wl = W.config(c)
    seed = int(wl["seed"])
    g = G.Pcmd(wl, separable=True)
    prms = wl["params"]
    n = len(prms)
    out = g.simulate(prms, seed=seed, want_raw=True, want_counts=True)
    fd = torch.empty((n, g.B, g.N, g.N), dtype=torch.float32, device="cuda")
    fc = torch.empty_like(fd)
    g.debug_taps(fd, fc)
    fast = g.simulate(prms, seed=seed, want_raw=True)                  # production kernel, as bench.py runs it
    g.debug_taps(None, None)
    H, st = g.hess(fast["mag"])
    data = np.concatenate([d.ravel() for d in wl["data_hess"]]).astype(np.uint32)
    lnl = g.loglike(H, st, torch.from_numpy(data.view(np.int32)).cuda()).cpu().numpy()
    torch.cuda.synchronize()
    assert g.status() == 0
    assert torch.equal(out["flux_raw"], fast["flux_raw"])
    assert torch.equal(out["mag"].view(torch.int32), fast["mag"].view(torch.int32))
    orc = O.Oracle(wl)
    stn = G.Pcmd.stats_to_numpy(st)
    for m in models:
        o = orc.simulate(prms[m], seed=seed, model=m)                  # the whole image
        w = g.debug_weights(m)
        assert np.array_equal(w["lam"], o["lam"])
        assert np.array_equal(out["total"][m].cpu().numpy().view(np.uint32), o["total"])      # every pixel
        assert np.array_equal(out["hash"][m].cpu().numpy().view(np.uint64), o["hash"])
        raw = fast["flux_raw"][m].cpu().numpy().reshape(g.B, -1)
        assert np.allclose(raw, o["F_raw"], rtol=FLUX_RTOL, atol=0)
        assert np.allclose(fd[m].cpu().numpy().reshape(g.B, -1), o["F_dust"], rtol=FLUX_RTOL, atol=0)
        assert np.allclose(fc[m].cpu().numpy().reshape(g.B, -1), o["G"], rtol=FLUX_RTOL, atol=0)
        mag = fast["mag"][m].cpu().numpy().reshape(g.B, -1)
        ok = ~np.isnan(o["mag"])
        assert np.array_equal(np.isnan(mag), ~ok)
        dmag = float(np.max(np.abs(mag[ok] - o["mag"][ok])))
        assert dmag <= MAG_ATOL
        off, parts = 0, []
        for hi, h in enumerate(wl["hess"]):
            nb = h["nx"] * h["ny"]
            Hg = H[m].cpu().numpy().view(np.uint32)[off:off + nb]
            off += nb
            moved, b64, b32, H64, s64 = hess_pixel_parity(orc, h, mag, o["mag"], Hg)
            parts.append((H64, b64, b32, moved))
            sg = stn[m, hi]
            assert int(Hg.sum()) + int(sg["n_out"]) + int(sg["n_bad"]) == g.P
            assert int(sg["n_bad"]) == s64["n_bad"]
            print("[c%d model %d hess %d] max |dmag| %.2e; %d of %d pixels moved bin, all within (%g, %g) mag of "
                  "an edge (oracle n_edge at 1e-5: %d)" % (c, m, hi, dmag, moved.size, g.P, EDGE_TOL_X, EDGE_TOL_Y,
                                                            s64["n_edge"]))
        lnl_poisson_parity(float(lnl[m]), parts, data, wl["like_floor"], "c%d model %d" % (c, m))
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
