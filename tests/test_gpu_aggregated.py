"""Aggregated sampler, sampler_mode = 1 (PAPER.md:75 footnote 3; DESIGN.md R-A1): CUDA path
against the oracle's orc_stage2_agg, element by element."""
import numpy as np
import pytest

from oracle import pcmd_oracle as O
from workloads import synthetic as W
from _parity import FLUX_RTOL, MAG_ATOL, hess_pixel_parity, lnl_poisson_parity

pytestmark = pytest.mark.gpu


def _agg(wl):
    return dict(wl, sampler_mode=1)


@pytest.mark.parametrize("cfg,n_im", [(1, 64), (2, 48), (3, 40), (4, 33), (5, 8)])
def test_aggregated_sampler_matches_the_oracle(cfg, n_im):
    """Star totals and the checksum over (point, count) bit-exact; flux 1e-5; magnitudes 1e-5 mag; Hess by the
    per-pixel edge rule; lnL 1e-4 -- the tolerances of the per-point sampler (north_star)."""
    import torch
    import paper_1904_00011_b200 as G
    wl = _agg(W.scaled(W.config(cfg), n_im))
    prms = wl["params"][:3]
    seed, m0 = 17, 2
    g = G.Pcmd(wl, separable=True)
    a = g.simulate(prms, seed=seed, model_index0=m0, want_raw=True, want_counts=True)
    fast = g.simulate(prms, seed=seed, model_index0=m0, want_raw=True)
    H, st = g.hess(fast["mag"])
    data = np.concatenate([d.ravel() for d in wl["data_hess"]]).astype(np.uint32)
    lnl = g.loglike(H, st, torch.from_numpy(data.view(np.int32)).cuda()).cpu().numpy()
    torch.cuda.synchronize()
    assert g.status() == 0
    assert torch.equal(a["flux_raw"], fast["flux_raw"])
    orc = O.Oracle(wl)
    for i, prm in enumerate(prms):
        o = orc.simulate(prm, seed=seed, model=m0 + i)
        assert o["total"].sum() > 0
        assert np.array_equal(a["total"][i].cpu().numpy().view(np.uint32), o["total"])
        assert np.array_equal(a["hash"][i].cpu().numpy().view(np.uint64), o["hash"])
        assert np.allclose(fast["flux_raw"][i].cpu().numpy().reshape(g.B, -1), o["F_raw"], rtol=FLUX_RTOL, atol=0)
        mag = fast["mag"][i].cpu().numpy().reshape(g.B, -1)
        ok = ~np.isnan(o["mag"])
        assert np.array_equal(np.isnan(mag), ~ok)
        assert np.max(np.abs(mag[ok] - o["mag"][ok])) <= MAG_ATOL
        off, parts = 0, []
        for h in wl["hess"]:
            nb = h["nx"] * h["ny"]
            moved, b64, b32, H64, _ = hess_pixel_parity(orc, h, mag, o["mag"], H[i].cpu().numpy().view(np.uint32)[off:off + nb])
            parts.append((H64, b64, b32, moved))
            off += nb
        lnl_poisson_parity(float(lnl[i]), parts, data, wl["like_floor"], "aggregated c%d model %d" % (cfg, i))
    g.close()


def test_aggregated_repeat_and_empty_model():
    import torch
    import paper_1904_00011_b200 as G
    wl = _agg(W.scaled(W.config(2), 24))
    g = G.Pcmd(wl, separable=True)
    prm = wl["params"][0]
    r = g.simulate_repeat(prm, 3, seed=5, model_index0=7, want_raw=True, want_counts=True)
    torch.cuda.synchronize()
    orc = O.Oracle(wl)
    for k in range(3):
        o = orc.simulate(prm, seed=5, model=7 + k)
        assert np.array_equal(r["total"][k].cpu().numpy().view(np.uint32), o["total"])
        assert np.array_equal(r["hash"][k].cpu().numpy().view(np.uint64), o["hash"])
    empty = dict(prm, sfh=np.zeros_like(prm["sfh"]))
    e = g.simulate([empty], seed=5, want_raw=True, want_counts=True)
    torch.cuda.synchronize()
    assert g.status() == 0 and not e["total"].any() and not e["flux_raw"].any()
    g.close()
