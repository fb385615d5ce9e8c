"""Repeated realisations of one parameter vector (Appendix A)."""
import numpy as np
import pytest

from workloads import synthetic as W

pytestmark = pytest.mark.gpu


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
