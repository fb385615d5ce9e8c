"""GPU edge cases: degenerate models, ragged and tiny images, the long-table fallback class, error
codes raised on the device.  Every comparison is against the CPU oracle on the same seeded inputs."""
import numpy as np
import pytest

from oracle import pcmd_oracle as O
from workloads import synthetic as W

pytestmark = pytest.mark.gpu


def _G():
    import paper_1904_00011_b200 as G
    return G


def _run(wl, prms=None, seed=3, separable=False):
    import torch
    G = _G()
    prms = prms or wl["params"]
    g = G.Pcmd(wl, separable=separable)
    out = g.simulate(prms, seed=seed, want_raw=True, want_counts=True)
    H, st = g.hess(out["mag"])
    torch.cuda.synchronize()
    res = dict(status=g.status(), g=g, total=out["total"].cpu().numpy().view(np.uint32),
               hash=out["hash"].cpu().numpy().view(np.uint64),
               raw=out["flux_raw"].cpu().numpy().reshape(len(prms), g.B, -1),
               mag=out["mag"].cpu().numpy().reshape(len(prms), g.B, -1),
               H=H.cpu().numpy().view(np.uint32), st=G.Pcmd.stats_to_numpy(st), Hdev=H, stdev=st)
    return res


@pytest.mark.parametrize("scale", [50.0, 2.0e3, 4.0e4])
def test_long_tables_every_search_class(scale):
    """lambda up to ~1e5: tables of 100s..1000s of thresholds (classes D7, D9 and the global-memory
    fallback), counts bit-exact, flux within 1e-5."""
    wl = W.tiny_model(n_im=12, J=12, B=2, seed=11, lam_scale=scale)
    orc = O.Oracle(wl)
    o = orc.simulate(wl["params"][0], seed=3)
    r = _run(wl)
    assert r["status"] == 0
    lens = r["g"].debug_weights(0)["len"]
    assert lens.max() > (31 if scale < 100 else (127 if scale < 1e4 else 511))
    assert np.array_equal(r["total"][0], o["total"]) and np.array_equal(r["hash"][0], o["hash"])
    assert np.allclose(r["raw"][0], o["F_raw"], rtol=1e-5, atol=0)
    ok = ~np.isnan(o["mag"])
    assert np.max(np.abs(r["mag"][0][ok] - o["mag"][ok])) <= 1e-5
    r["g"].close()


def test_no_stars_at_all_gives_nan_magnitudes_and_minus_inf_lnl():
    import torch
    wl = W.tiny_model(n_im=8, J=8)
    prm = dict(wl["params"][0], sfh=np.zeros(1))
    r = _run(wl, [prm])
    assert r["status"] == 0
    assert not r["total"].any() and not r["raw"].any()
    assert np.isnan(r["mag"]).all()
    assert r["st"][0, 0]["n_bad"] == 64 and not r["H"].any()
    data = torch.ones(r["g"].bins_total, dtype=torch.int32, device="cuda")
    lnl = r["g"].loglike(r["Hdev"], r["stdev"], data).cpu().numpy()
    assert lnl[0] == -np.inf
    r["g"].close()


def test_lambda_above_2_pow_22_raises_erange_on_the_device():
    wl = W.tiny_model(n_im=4, J=8)
    prm = dict(wl["params"][0], sfh=np.array([1.0e9]))
    r = _run(wl, [prm])
    assert r["status"] == -2        # PCMD_ERANGE
    r["g"].close()


@pytest.mark.parametrize("n_im", [1, 3, 33])
def test_tiny_and_ragged_images(n_im):
    """Images smaller than a tile, smaller than the PSF, and not a multiple of any tile size."""
    wl = W.scaled(W.config(2), n_im)
    orc = O.Oracle(wl)
    o = orc.simulate(wl["params"][0], seed=3)
    for sep in (False, True):
        r = _run(wl, seed=3, separable=sep)
        assert r["status"] == 0
        assert np.array_equal(r["total"][0], o["total"]) and np.array_equal(r["hash"][0], o["hash"])
        assert np.allclose(r["raw"][0], o["F_raw"], rtol=1e-5, atol=0)
        ok = ~np.isnan(o["mag"])
        assert np.array_equal(np.isnan(r["mag"][0]), np.isnan(o["mag"]))
        assert np.max(np.abs(r["mag"][0][ok] - o["mag"][ok])) <= 1e-5
        H32, _ = orc.hess_f32(wl["hess"][0], r["mag"][0])
        assert np.array_equal(r["H"][0].reshape(H32.shape), H32)
        r["g"].close()


def test_delta_psf_is_the_identity_and_model_index_changes_the_stream():
    import torch
    G = _G()
    wl = W.with_psf(W.scaled(W.config(1), 16), 1, [1.0, 1.0])
    wl["read_sigma"] = np.zeros(2)           # noise off: mag = zp - 2.5 log10(F)
    g = G.Pcmd(wl)
    a = g.simulate(wl["params"], seed=5, model_index0=0, want_raw=True)
    b = g.simulate(wl["params"], seed=5, model_index0=1, want_raw=True)
    torch.cuda.synchronize()
    Fa, Fb = a["flux_raw"].cpu().numpy(), b["flux_raw"].cpu().numpy()
    assert not np.array_equal(Fa, Fb)
    orc = O.Oracle(wl)
    o1 = orc.simulate(wl["params"][0], seed=5, model=1)
    assert np.allclose(Fb.reshape(2, -1), o1["F_raw"], rtol=1e-5, atol=0)
    want = wl["zp"][:, None] - 2.5 * np.log10(Fa.reshape(2, -1).astype(np.float64))
    got = a["mag"].cpu().numpy().reshape(2, -1)
    ok = np.isfinite(want)
    assert np.max(np.abs(got[ok] - want[ok])) <= 1e-5
    g.close()


def test_bad_arguments_are_rejected_without_touching_the_device():
    import ctypes as C
    G = _G()
    wl = W.tiny_model(n_im=4, J=8)
    g = G.Pcmd(wl)
    L = G.lib()
    assert L.pcmd_simulate(g._ctx, None, 1, C.c_uint64(0), 0, None, None, None, None, None) == -1
    assert L.pcmd_hess(g._ctx, None, 1, None, None, None) == -1
    assert L.pcmd_loglike(g._ctx, None, None, 1, None, None, 0, None, None) == -1
    with pytest.raises(G.PcmdError):
        g.simulate([dict(wl["params"][0], feh_sigma=0.0)])
    with pytest.raises(G.PcmdError):
        g.simulate([dict(wl["params"][0], sfh=np.array([-1.0]))])
    g.close()


@pytest.mark.parametrize("c,n_im,G", [(3, 40, 4), (2, 48, 3), (1, 64, 4), (2, 7, 4)])
def test_subpixel_psf_grid(c, n_im, G):
    """PAPER.md:180 (R-Q19): G x G shifted PSFs, an output pixel uses the PSF of its cell; cells that
    do not line up with the 32 x 32 CUDA tiles, and an image smaller than a cell row."""
    import torch
    Gm = _G()
    wl = W.with_psf_grid(W.scaled(W.config(c), n_im), G)
    orc = O.Oracle(wl)
    o = orc.simulate(wl["params"][0], seed=2)
    g = Gm.Pcmd(wl)
    fc = torch.empty((1, g.B, g.N, g.N), dtype=torch.float32, device="cuda")
    g.debug_taps(None, fc)
    out = g.simulate(wl["params"][:1], seed=2)
    torch.cuda.synchronize()
    assert g.status() == 0
    assert np.allclose(fc.cpu().numpy().reshape(g.B, -1), o["G"], rtol=1e-5, atol=0)
    mag = out["mag"].cpu().numpy().reshape(g.B, -1)
    ok = ~np.isnan(o["mag"])
    assert np.array_equal(np.isnan(mag), ~ok)
    assert np.max(np.abs(mag[ok] - o["mag"][ok])) <= 1e-5
    # and it is not the un-shifted PSF's answer
    o1 = O.Oracle(W.scaled(W.config(c), n_im)).stage4(o["F_dust"])
    assert not np.allclose(o1, o["G"], rtol=1e-4, atol=0)
    g.close()
    with pytest.raises(ValueError):
        Gm.Pcmd(wl, separable=True)


def test_capped_arena_non_power_of_two_batch():
    """50 <= n_models < 799 at J = 10 500 caps the per-model arena of padded search tables at 2^28 / n_models
    words; every model's arena must still start 16-byte aligned for the bulk copies (a batch that is not a
    power of two used to leave model 1 misaligned).  All models against the oracle."""
    wl = W.scaled(W.config(4), 32)
    base = wl["params"]
    prms = [base[i % len(base)] for i in range(50)]
    # make some models D-class heavy so that the arena is really read
    for i in (1, 7, 49):
        prms[i] = dict(prms[i], sfh=np.asarray(prms[i]["sfh"]) * 40.0)
    r = _run(wl, prms, seed=5, separable=True)
    assert r["status"] == 0
    orc = O.Oracle(wl)
    for i in (0, 1, 7, 23, 49):
        o = orc.simulate(prms[i], seed=5, model=i)
        assert np.array_equal(r["total"][i], o["total"]) and np.array_equal(r["hash"][i], o["hash"])
        assert np.allclose(r["raw"][i], o["F_raw"], rtol=1e-5, atol=0)
    r["g"].close()


def test_pipe_bench_reports_sane_rates():
    """pcmd_pipe_bench (measurement support, csrc/pipes.cu): every stream runs and reports a rate between 0 and 2
    warp-instructions per clock per scheduler; the Philox-only kernel lands between 1e12 and 2.4e12 draws/s on a B200."""
    G = _G()
    rows = G.pipe_bench(iters=512)
    assert len(rows) >= 10 and all(0.0 < r["rate"] < 2.0 and r["ms"] > 0 for r in rows)
    ph = [r for r in rows if r["name"].startswith("Philox4x32-10")][0]
    assert 1.0e12 < 4.0 * ph["steps_per_s"] < 2.4e12
    one = G.pipe_bench(iters=512, only="LOP3 (xor3)")
    assert len(one) == 1 and 0.4 < one[0]["rate"] < 0.6
