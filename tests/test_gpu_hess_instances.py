"""Stage 6 alone on synthetic magnitudes, through every instance of k_hess (csrc/hess_like.cu): 512-thread blocks with a
shared-memory histogram, the 1024-thread instance (histogram > 100 KB), the global-atomics instance (> 200 KB), one
block per diagram and several, the 16-byte-load path and the scalar one (pixel count not a multiple of four), with
NaN and out-of-window pixels (the two spare counters of the branch-free binning).  Against the oracle's Hess taken in
the kernel's precision (orc_hess_f32: bit-exact counts, R-Q13).  PAPER.md:57,130,218."""
import numpy as np
import pytest

from oracle import pcmd_oracle as O
from workloads import synthetic as W

pytestmark = pytest.mark.gpu


@pytest.mark.parametrize("n_im,nbin,n_models", [
    (64, 100, 1),        # one block per diagram (4096 px), 512 threads, shared histogram
    (160, 100, 2),       # several blocks per diagram: memset + atomics flush + k_hess_stats
    (160, 190, 2),       # 144 KB histogram: the 1024-thread instance, several blocks
    (64, 240, 3),        # 230 KB histogram: global atomics
    (33, 100, 2),        # 1089 px: not a multiple of four, scalar loads
    (32, 100, 700)])     # a GPU-filling batch: one block per diagram, plain stores
def test_hess_instances_against_oracle(n_im, nbin, n_models):
    import torch
    import paper_1904_00011_b200 as G
    from paper_1904_00011_b200 import binding
    wl = dict(W.scaled(W.config(3), n_im))
    wl["hess"] = [dict(h, nx=nbin, ny=nbin) for h in wl["hess"]]
    wl.pop("data_hess", None); wl.pop("data_stats", None)
    g = G.Pcmd(wl)
    orc = O.Oracle(wl)
    P = g.P
    rng = np.random.default_rng(1000 * n_im + nbin)
    h0 = wl["hess"][0]
    # magnitudes around the window: ~70 % of the pixels inside, the rest above, below, left or right of it
    y = rng.uniform(h0["y_lo"] - 0.15, h0["y_hi"] + 0.15, size=(n_models, 1, P))
    col = rng.uniform(-0.7, 0.45, size=(n_models, 2, P))
    mag = np.concatenate([y + col, y], axis=1).astype(np.float32)            # bands 0, 1 = y + colour; band 2 = y
    mag[:, 0, ::17] = np.nan
    mag[:, 2, 5::29] = np.nan
    mag[-1, 1, :] = np.nan                                                   # a diagram with no valid pixel at all
    tm = torch.from_numpy(mag.reshape(n_models, 3, n_im, n_im)).cuda()
    H, st = g.hess(tm)
    torch.cuda.synchronize()
    Hn = H.cpu().numpy().view(np.uint32)
    stn = st.cpu().numpy().view(binding.STATS_DTYPE).reshape(n_models, len(wl["hess"]))
    for i in sorted({0, n_models // 2, n_models - 1}):
        off = 0
        for hi, h in enumerate(wl["hess"]):
            nb = h["nx"] * h["ny"]
            H32, s32 = orc.hess_f32(h, mag[i])
            assert np.array_equal(Hn[i, off:off + nb].reshape(h["ny"], h["nx"]), H32)
            off += nb
            sg = stn[i, hi]
            assert (int(sg["n_in"]), int(sg["n_out"]), int(sg["n_bad"])) == (s32["n_in"], s32["n_out"], s32["n_bad"])
            assert int(sg["n_in"]) + int(sg["n_out"]) + int(sg["n_bad"]) == P
            assert abs(sg["sum_x"] - s32["sum_x"]) <= 1e-9 * max(1.0, abs(s32["sum_x"]))
            assert abs(sg["sum_y"] - s32["sum_y"]) <= 1e-9 * max(1.0, abs(s32["sum_y"]))
    assert int(stn[0, 0]["n_in"]) > P // 3 and int(stn[0, 0]["n_bad"]) > 0 and int(stn[0, 0]["n_out"]) > 0
    assert int(stn[-1, 1]["n_bad"]) == P and int(stn[-1, 1]["n_in"]) == 0
    g.close()
