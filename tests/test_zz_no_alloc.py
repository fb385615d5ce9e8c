"""pcmd_hess_noalloc (include/pcmd.h): stage 6 with its scratch in a fixed device array of the library instead
of the ctx's grow-on-demand buffer, for callers that must not allocate.  Checked against the existing path
(pcmd_hess) on two calls in a row that share the array: diagrams and statistics bit-identical (same kernels, same
launch geometry; the Hess is integer work: the suite's bar for it is exact).  Collected last on purpose (the file
name): the run uses -x."""
import numpy as np
import pytest

from workloads import synthetic as W

pytestmark = pytest.mark.gpu

MAX_PARTS = 8192            # PCMD_HESS_NOALLOC_MAX_PARTS
ELIMIT = -5


def _both(g, mag):
    import torch
    n = mag.shape[0]
    H0, S0 = g.hess(mag)
    H1 = torch.full((n, g.bins_total), -1, dtype=torch.int32, device="cuda")          # overwritten, whatever it held
    S1 = torch.full((n, len(g.hess_specs), 4), -1.0, dtype=torch.float64, device="cuda")
    g.hess_noalloc(mag, H1, S1)
    torch.cuda.synchronize()
    assert g.status() == 0
    return H0, S0, H1, S1


def test_noalloc_hess_matches_existing_path_on_two_calls_in_a_row():
    import torch
    import paper_1904_00011_b200 as G
    from paper_1904_00011_b200 import binding
    assert binding.lib().pcmd_hess_noalloc_setup() == 0
    wl = W.scaled(W.config(3), 256)                      # c3's three bands and two diagrams, 256 x 256 pixels
    g = G.Pcmd(wl)
    prm = [dict(wl["params"][0])]
    # call 1: one model, 16 blocks per diagram (partials + the statistics kernel read the fixed array)
    mag1 = g.simulate(prm, seed=11)["mag"]
    assert g.hess_noalloc_parts(1) == 2 * 16
    H0, S0, H1, S1 = _both(g, mag1)
    assert int(H0.sum()) > 0
    assert torch.equal(H0, H1)
    assert torch.equal(S0.view(torch.int64), S1.view(torch.int64))
    # call 2, straight after: other magnitudes, another batch size (another partition of the same array, which
    # still holds call 1's partials), some NaN and out-of-window pixels
    mag2 = g.simulate([prm[0]] * 3, seed=12, model_index0=7)["mag"].clone()
    mag2[1, 0, ::5, ::3] = float("nan")
    mag2[2] += 30.0
    H0, S0, H1, S1 = _both(g, mag2)
    assert torch.equal(H0, H1)
    assert torch.equal(S0.view(torch.int64), S1.view(torch.int64))
    st = S1.cpu().numpy().view(binding.STATS_DTYPE).reshape(3, -1)
    assert int(st["n_bad"][1][0]) > 0 and int(st["n_bad"][1][1]) == 0 and int(st["n_in"][2].max()) == 0
    assert np.all(st["n_in"].astype(np.int64) + st["n_out"] + st["n_bad"] == g.P)
    # without statistics (the single-block branch then writes its partial into the array)
    H2 = torch.empty_like(H1)
    g.hess_noalloc(mag2, H2, None)
    torch.cuda.synchronize()
    assert torch.equal(H0, H2)
    g.close()


def test_noalloc_hess_one_block_per_diagram_and_the_size_limit():
    import torch
    import paper_1904_00011_b200 as G
    wl = W.scaled(W.config(4), 32)                       # 32 x 32 pixels, 2 bands, one diagram
    g = G.Pcmd(wl)
    n_hess = len(g.hess_specs)
    spec = g.hess_specs[0]
    gen = torch.Generator(device="cuda").manual_seed(5)
    for n in (1500, MAX_PARTS // n_hess):                # a GPU-filling batch: one block per diagram; the largest legal one
        assert g.hess_noalloc_parts(n) == n * n_hess <= MAX_PARTS
        mag = torch.rand((n, g.B, g.N, g.N), generator=gen, device="cuda") * (spec["y_hi"] - spec["y_lo"]) + spec["y_lo"]
        H0, S0, H1, S1 = _both(g, mag)
        assert torch.equal(H0, H1)
        assert torch.equal(S0.view(torch.int64), S1.view(torch.int64))
    # one model more than the fixed array holds: refused before anything is launched, outputs untouched
    n = MAX_PARTS // n_hess + 1
    mag = torch.zeros((n, g.B, g.N, g.N), device="cuda")
    H = torch.full((n, g.bins_total), -7, dtype=torch.int32, device="cuda")
    launches = g.launch_count()
    with pytest.raises(G.PcmdError) as ei:
        g.hess_noalloc(mag, H, None)
    assert ei.value.code == ELIMIT and "no-allocation" in str(ei.value)
    torch.cuda.synchronize()
    assert g.launch_count() == launches and int((H != -7).sum()) == 0
    g.close()
