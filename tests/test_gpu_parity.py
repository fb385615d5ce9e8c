"""GPU parity: the CUDA path (through the C ABI) against the CPU oracle, element by element, on
the same seeded inputs.  Tolerances are north_star's: counts bit-exact, fluxes 1e-5 relative,
magnitudes 1e-5 mag, Hess bins differ only through pixels within 1e-5 mag of a bin edge,
lnL 1e-4 relative."""
import numpy as np
import pytest

from oracle import pcmd_oracle as O
from workloads import synthetic as W
from _parity import (EDGE_TOL_X, EDGE_TOL_Y, FLUX_RTOL, LNL_RTOL, MAG_ATOL, hess_pixel_parity,
                     lnl_poisson_parity, rebin_moved, restat_moved)

pytestmark = pytest.mark.gpu


def _gpu():
    import paper_1904_00011_b200 as G
    return G


def _cases():
    c1 = W.config(1)
    c2 = W.scaled(W.config(2), 48)
    c3 = W.scaled(W.config(3), 40)          # ragged: 40 is not a multiple of the 32-wide tiles
    c3m2 = dict(c3, dust_mode=2, name="c3m2@40")
    c4 = W.scaled(W.config(4), 32)
    c4["params"] = c4["params"][:5]
    c5 = W.scaled(W.config(5), 24)
    return {"c1": c1, "c2": c2, "c3": c3, "c3m2": c3m2, "c4": c4, "c5": c5}


CASES = _cases()


@pytest.fixture(scope="module", params=list(CASES))
def run(request):
    """Runs the oracle and the GPU path once per case, with every intermediate."""
    import torch
    G = _gpu()
    wl = CASES[request.param]
    seed = int(wl["seed"])
    orc = O.Oracle(wl)
    osim = [orc.simulate(p, seed=seed, model=i) for i, p in enumerate(wl["params"])]
    g = G.Pcmd(wl)
    n = len(wl["params"])
    fd = torch.empty((n, g.B, g.N, g.N), dtype=torch.float32, device="cuda")
    fc = torch.empty_like(fd)
    g.debug_taps(fd, fc)
    out = g.simulate(wl["params"], seed=seed, want_raw=True, want_counts=True)
    assert g.status() == 0
    w = [g.debug_weights(i) for i in range(n)]
    g.debug_taps(None, None)
    fast = g.simulate(wl["params"], seed=seed, want_raw=True)
    H, st = g.hess(out["mag"])
    torch.cuda.synchronize()
    res = dict(wl=wl, orc=orc, osim=osim, g=g, n=n, w=w,
               mag=out["mag"].cpu().numpy().reshape(n, g.B, -1).astype(np.float32),
               raw=out["flux_raw"].cpu().numpy().reshape(n, g.B, -1),
               raw_fast=fast["flux_raw"].cpu().numpy().reshape(n, g.B, -1),
               mag_fast=fast["mag"].cpu().numpy().reshape(n, g.B, -1),
               hash=out["hash"].cpu().numpy().view(np.uint64), total=out["total"].cpu().numpy().view(np.uint32),
               fd=fd.cpu().numpy().reshape(n, g.B, -1), fc=fc.cpu().numpy().reshape(n, g.B, -1),
               H=H.cpu().numpy().view(np.uint32), st=G.Pcmd.stats_to_numpy(st), Hdev=H, stdev=st)
    yield res
    g.close()


def test_stage1_lambda_and_tables_bit_exact(run):
    for i in range(run["n"]):
        o, w = run["osim"][i], run["w"][i]
        assert np.array_equal(w["lam"], o["lam"])                       # fp64 bit-equal
        assert np.allclose(w["flux"], o["flux"], rtol=2e-7, atol=0)     # fp32 rounding of the fp64 flux
        pos = 0
        for j in range(0, run["orc"].J, max(1, run["orc"].J // 400)):   # a spread of points, full tables
            T, k_lo, k_hi = O.poisson_table(float(o["lam"][j]))
            stored = T[(T > 0) & (T < 2 ** 32)]
            k0 = k_lo + int(np.count_nonzero(T == 0)) if o["lam"][j] > 0 else 0
            off = int(w["len"][:j].sum())
            if o["lam"][j] > 0:
                assert w["k0"][j] == k0 and w["len"][j] == stored.size
                assert np.array_equal(w["tables"][off:off + stored.size].astype(np.uint64), stored)
            else:
                assert w["len"][j] == 0
            pos += 1
        assert pos > 0


def test_stage2_counts_bit_exact_and_flux(run):
    for i in range(run["n"]):
        o = run["osim"][i]
        assert np.array_equal(run["total"][i], o["total"])
        assert np.array_equal(run["hash"][i], o["hash"])
        assert np.allclose(run["raw"][i], o["F_raw"], rtol=FLUX_RTOL, atol=0)
    # the production kernel (no count tracking) produces the very same fluxes and magnitudes
    assert np.array_equal(run["raw"], run["raw_fast"])
    assert np.array_equal(run["mag"], run["mag_fast"], equal_nan=True)


def test_stage3_dust_and_stage4_conv(run):
    for i in range(run["n"]):
        o = run["osim"][i]
        assert np.allclose(run["fd"][i], o["F_dust"], rtol=FLUX_RTOL, atol=0)
        assert np.allclose(run["fc"][i], o["G"], rtol=FLUX_RTOL, atol=0)


def test_stage5_magnitudes(run):
    for i in range(run["n"]):
        o = run["osim"][i]
        assert np.array_equal(np.isnan(run["mag"][i]), np.isnan(o["mag"]))
        ok = ~np.isnan(o["mag"])
        assert np.max(np.abs(run["mag"][i][ok] - o["mag"][ok])) <= MAG_ATOL


def test_stage6_hess(run):
    wl, orc = run["wl"], run["orc"]
    for i in range(run["n"]):
        off = 0
        for hi, h in enumerate(wl["hess"]):
            nb = h["nx"] * h["ny"]
            Hg = run["H"][i, off:off + nb].reshape(h["ny"], h["nx"])
            off += nb
            # (a) same decision in the kernel's precision on the kernel's magnitudes: bit-exact
            H32, s32 = orc.hess_f32(h, run["mag"][i])
            assert np.array_equal(Hg, H32)
            sg = run["st"][i, hi]
            assert (sg["n_in"], sg["n_out"], sg["n_bad"]) == (s32["n_in"], s32["n_out"], s32["n_bad"])
            assert abs(sg["sum_x"] - s32["sum_x"]) <= 1e-9 * max(1.0, abs(s32["sum_x"]))
            assert abs(sg["sum_y"] - s32["sum_y"]) <= 1e-9 * max(1.0, abs(s32["sum_y"]))
            assert int(Hg.sum()) + int(sg["n_out"]) + int(sg["n_bad"]) == orc.P
            # (b) against the fp64 oracle end to end, pixel by pixel: a pixel may change bin only if the oracle
            # flags it within 1e-5 mag of a y edge or 2e-5 mag of a colour edge (tests/_parity.py)
            moved, _, _, _, _ = hess_pixel_parity(orc, h, run["mag"][i], run["osim"][i]["mag"], Hg)
            print("[%s model %d hess %d] %d pixels moved bin (all flagged near an edge)" % (wl["name"], i, hi, moved.size))


def test_stage7_loglike(run):
    import torch
    G = _gpu()
    wl, orc, g = run["wl"], run["orc"], run["g"]
    if wl.get("data_hess") is None:
        pytest.skip("no frozen data Hess")
    data = np.concatenate([d.ravel() for d in wl["data_hess"]]).astype(np.uint32)
    dd = torch.from_numpy(data.view(np.int32)).cuda()
    ds = np.zeros(len(wl["hess"]), dtype=G.binding.STATS_DTYPE)
    for hi, s in enumerate(wl["data_stats"]):
        for k in ("n_in", "n_out", "n_bad", "sum_x", "sum_y"):
            ds[hi][k] = s[k]
    dsd = torch.from_numpy(ds.view(np.float64).reshape(len(wl["hess"]), 4)).cuda()
    for mode, literal in ((G.LIKE_POISSON, None), (G.LIKE_GAUSS, False), (G.LIKE_GAUSS_LITERAL, True)):
        lg = g.loglike(run["Hdev"], run["stdev"], dd, dsd, mode=mode).cpu().numpy()
        for i in range(run["n"]):
            want_iso, want_e2e, off, eq4_slack = 0.0, 0.0, 0, 0.0
            for hi, h in enumerate(wl["hess"]):
                nb = h["nx"] * h["ny"]
                Hg = run["H"][i, off:off + nb]
                H64, s64 = orc.hess(h, run["osim"][i]["mag"])
                d = data[off:off + nb]
                off += nb
                if literal is None:
                    want_iso += O.loglike_poisson(Hg, d, wl["like_floor"])
                    want_e2e += O.loglike_poisson(H64, d, wl["like_floor"])
                else:
                    sg = {k: run["st"][i, hi][k] for k in ("n_in", "n_out", "n_bad", "sum_x", "sum_y")}
                    want_iso += O.loglike_gauss(Hg, sg, d, wl["data_stats"][hi], literal)
                    want_e2e += O.loglike_gauss(H64, s64, d, wl["data_stats"][hi], literal)
                    sd = wl["data_stats"][hi]
                    if s64["n_in"] == 0:
                        continue
                    dC = abs(sd["sum_x"] / sd["n_in"] - s64["sum_x"] / s64["n_in"])
                    dM = abs(sd["sum_y"] / sd["n_in"] - s64["sum_y"] / s64["n_in"])
                    eq4_slack += (dC + dM + MAG_ATOL) * MAG_ATOL / 0.05 ** 2
            if not np.isfinite(want_iso):       # a model with no pixel inside the data window: -inf on both sides
                assert lg[i] == want_iso
                continue
            assert abs(lg[i] - want_iso) <= 1e-10 * abs(want_iso)        # stage-isolated
            # end to end (north_star 1e-4): moved edge pixels re-binned the GPU's way, never skipped
            off, parts = 0, []
            for hi, h in enumerate(wl["hess"]):
                nb = h["nx"] * h["ny"]
                moved, b64, b32, H64, s64 = hess_pixel_parity(orc, h, run["mag"][i], run["osim"][i]["mag"],
                                                              run["H"][i, off:off + nb])
                parts.append((H64, b64, b32, moved, s64))
                off += nb
            if literal is None:
                lnl_poisson_parity(float(lg[i]), [q[:4] for q in parts], data, wl["like_floor"],
                                   "%s model %d" % (wl["name"], i))
            else:
                # Eq. 4's term (dC^2 + dM^2) / (2 * 0.05^2) moves with the fp32 magnitudes (<= MAG_ATOL each):
                # |d lnL| <= (|dC| + |dM| + MAG_ATOL) MAG_ATOL / 0.05^2
                want, off = 0.0, 0
                for hi, (H64, b64, b32, moved, s64) in enumerate(parts):
                    nb = H64.size
                    Hr = rebin_moved(H64, b64, b32, moved) if moved.size else H64
                    s_use = restat_moved(s64, wl["hess"][hi], run["osim"][i]["mag"], b64, b32, moved)
                    want += O.loglike_gauss(Hr, s_use, data[off:off + nb], wl["data_stats"][hi], literal)
                    off += nb
                err = abs(lg[i] - want)
                bound = LNL_RTOL * abs(want) + eq4_slack
                print("[lnL Gauss%s %s model %d] |dlnL| observed %.3e, bound %.3e (of which Eq. 4 slack %.3e)" % (
                    " literal" if literal else "", wl["name"], i, err, bound, eq4_slack))
                assert err <= bound
    # host-buffer entry point = the same three calls
    lnl, Hh, sth = g.evaluate_host(wl["params"], data, seed=int(wl["seed"]))
    assert np.array_equal(Hh, run["H"])
    lg = g.loglike(run["Hdev"], run["stdev"], dd, dsd, mode=G.LIKE_POISSON).cpu().numpy()
    assert np.array_equal(lnl, lg)


@pytest.mark.parametrize("name", ["c2", "c3", "c5"])
def test_separable_psf_path(name):
    """psf_separable=1 (row and column factors, fused row/column passes) against the oracle's 2-D sum."""
    import torch
    G = _gpu()
    wl = CASES[name]
    seed = int(wl["seed"])
    orc = O.Oracle(wl)
    o = orc.simulate(wl["params"][0], seed=seed)
    g = G.Pcmd(wl, separable=True)
    fc = torch.empty((1, g.B, g.N, g.N), dtype=torch.float32, device="cuda")
    g.debug_taps(None, fc)
    out = g.simulate(wl["params"][:1], seed=seed)
    torch.cuda.synchronize()
    assert g.status() == 0
    assert np.allclose(fc.cpu().numpy().reshape(g.B, -1), o["G"], rtol=FLUX_RTOL, atol=0)
    mag = out["mag"].cpu().numpy().reshape(g.B, -1)
    ok = ~np.isnan(o["mag"])
    assert np.array_equal(np.isnan(mag), np.isnan(o["mag"]))
    assert np.max(np.abs(mag[ok] - o["mag"][ok])) <= MAG_ATOL
    g.close()
