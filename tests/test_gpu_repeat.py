"""Repeated realisations of one parameter vector (Appendix A)."""
import numpy as np
import pytest

from oracle import pcmd_oracle as O
from workloads import synthetic as W
from _parity import FLUX_RTOL, MAG_ATOL, hess_pixel_parity, lnl_poisson_parity

pytestmark = pytest.mark.gpu


def test_repeat_realisation_r_is_the_oracle_model_index0_plus_r():
    """PAPER.md:385 (App. A: the best-fit likelihood recomputed many times): realisation r of
    pcmd_simulate_repeat is, element by element, Oracle.simulate(prm, seed, model=model_index0 + r):
    counts bit-exact, flux 1e-5, magnitudes 1e-5 mag, Hess by the per-pixel edge rule, lnL 1e-4."""
    import torch
    import paper_1904_00011_b200 as G
    wl = W.scaled(W.config(3), 56)
    g = G.Pcmd(wl, separable=True)
    prm, seed, m0, R = wl["params"][0], 9, 3, 4
    a = g.simulate_repeat(prm, R, seed=seed, model_index0=m0, want_raw=True, want_counts=True)
    fast = g.simulate_repeat(prm, R, seed=seed, model_index0=m0, want_raw=True)     # production kernel
    H, st = g.hess(fast["mag"])
    data = np.concatenate([d.ravel() for d in wl["data_hess"]]).astype(np.uint32)
    lnl = g.loglike(H, st, torch.from_numpy(data.view(np.int32)).cuda()).cpu().numpy()
    torch.cuda.synchronize()
    assert g.status() == 0
    assert torch.equal(a["flux_raw"], fast["flux_raw"])
    orc = O.Oracle(wl)
    for r in range(R):
        o = orc.simulate(prm, seed=seed, model=m0 + r)
        assert np.array_equal(a["total"][r].cpu().numpy().view(np.uint32), o["total"])
        assert np.array_equal(a["hash"][r].cpu().numpy().view(np.uint64), o["hash"])
        assert np.allclose(fast["flux_raw"][r].cpu().numpy().reshape(g.B, -1), o["F_raw"], rtol=FLUX_RTOL, atol=0)
        mag = fast["mag"][r].cpu().numpy().reshape(g.B, -1)
        ok = ~np.isnan(o["mag"])
        assert np.array_equal(np.isnan(mag), ~ok)
        assert np.max(np.abs(mag[ok] - o["mag"][ok])) <= MAG_ATOL
        off, parts = 0, []
        for h in wl["hess"]:
            nb = h["nx"] * h["ny"]
            moved, b64, b32, H64, _ = hess_pixel_parity(orc, h, mag, o["mag"], H[r].cpu().numpy().view(np.uint32)[off:off + nb])
            parts.append((H64, b64, b32, moved))
            off += nb
        lnl_poisson_parity(float(lnl[r]), parts, data, wl["like_floor"], "repeat r=%d" % r)
    g.close()


def test_repeat_equals_a_batch_of_copies_bit_for_bit():
    import torch
    import paper_1904_00011_b200 as G
    wl = W.scaled(W.config(3), 40)
    g = G.Pcmd(wl, separable=True)
    prm = wl["params"][0]
    a = g.simulate_repeat(prm, 5, seed=9, model_index0=3, want_raw=True)
    b = g.simulate([prm] * 5, seed=9, model_index0=3, want_raw=True)
    torch.cuda.synchronize()
    assert g.status() == 0
    assert torch.equal(a["flux_raw"], b["flux_raw"])
    assert torch.equal(a["mag"].view(torch.int32), b["mag"].view(torch.int32))
    # realisations differ from one another
    assert not torch.equal(a["flux_raw"][0], a["flux_raw"][1])
    g.close()


def test_likelihood_scatter_over_seeds_shrinks_with_image_size():
    """the likelihood is stochastic and its variance decreases with N_im."""
    import torch
    import paper_1904_00011_b200 as G
    full = W.config(2)
    data = np.concatenate([d.ravel() for d in full["data_hess"]]).astype(np.uint32)
    dd = torch.from_numpy(data.view(np.int32)).cuda()
    sd = {}
    for n_im in (48, 192):
        wl = W.scaled(full, n_im)
        g = G.Pcmd(wl, separable=True)
        out = g.simulate_repeat(wl["params"][0], 24, seed=4)
        H, st = g.hess(out["mag"])
        lnl = g.loglike(H, st, dd).cpu().numpy()
        assert np.all(np.isfinite(lnl)) and np.unique(lnl).size == 24
        sd[n_im] = float(np.std(lnl))
        g.close()
    assert sd[192] < 0.7 * sd[48]
