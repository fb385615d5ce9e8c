"""Shared assertions of the GPU parity tests (north_star tolerances).

Hess (north_star: "Hess bins may differ only for pixels lying within 1e-5 mag of a bin edge"): the check is
per pixel.  The bin of pixel p on the GPU side is the kernel-precision decision on the GPU's magnitudes
(orc_hess_pixels_f32, whose histogram must be the GPU Hess bit for bit); on the oracle side it is the fp64
decision on the oracle's magnitudes.  Every pixel whose two bins differ must carry the oracle's near-edge
flag: magnitude within EDGE_TOL_Y = 1e-5 of a y edge, or colour within EDGE_TOL_X = 2e-5 of an x edge (a
colour is the difference of two magnitudes, each allowed 1e-5; DESIGN.md R-Q17).

lnL (north_star: 1e-4 relative): end to end against the oracle's own Hess when no pixel moved;
when pixels moved (all of them verified to be edge pixels), those pixels -- and only those -- are re-binned
the GPU's way in the oracle's Hess and the 1e-4 bar is applied against that.  Nothing is skipped silently:
the number of moved pixels and the raw end-to-end difference are printed.
"""
import numpy as np

from oracle import pcmd_oracle as O

FLUX_RTOL = 1e-5
MAG_ATOL = 1e-5
LNL_RTOL = 1e-4
EDGE_TOL_X = 2e-5
EDGE_TOL_Y = 1e-5


def hess_pixel_parity(orc, h, mag_gpu, mag_orc, H_gpu):
    """Asserts the per-pixel edge-membership rule for one Hess spec.  Returns (moved pixel indices,
    oracle per-pixel bins, GPU per-pixel bins, oracle fp64 Hess, oracle stats)."""
    nb = h["nx"] * h["ny"]
    b32 = orc.hess_pixels_f32(h, mag_gpu)
    Hg = np.asarray(H_gpu).reshape(-1)
    assert np.array_equal(np.bincount(b32[b32 >= 0], minlength=nb).astype(np.uint32), Hg), \
        "GPU Hess is not the kernel-precision histogram of the GPU magnitudes"
    b64, near = orc.hess_pixels(h, mag_orc, tol_x=EDGE_TOL_X, tol_y=EDGE_TOL_Y)
    H64, s64 = orc.hess(h, mag_orc, edge_tol=EDGE_TOL_Y, want_edges=True)
    assert np.array_equal(np.bincount(b64[b64 >= 0], minlength=nb).astype(np.uint32), H64.ravel())
    moved = np.nonzero(b32 != b64)[0]
    bad = moved[near[moved] == 0]
    assert bad.size == 0, "%d pixels changed bin without lying within (%g, %g) mag of a bin edge, e.g. pixel %d" % (
        bad.size, EDGE_TOL_X, EDGE_TOL_Y, int(bad[0]) if bad.size else -1)
    # NaN pattern: a pixel that is bad on one side is bad on the other (magnitudes are compared separately)
    assert np.array_equal(b32 == -2, b64 == -2)
    return moved, b64, b32, H64, s64


def rebin_moved(H64, b64, b32, moved):
    """The oracle's Hess with exactly the moved pixels re-binned the GPU's way."""
    H = H64.astype(np.int64).ravel().copy()
    for p in moved:
        if b64[p] >= 0:
            H[b64[p]] -= 1
        if b32[p] >= 0:
            H[b32[p]] += 1
    assert H.min() >= 0
    return H.astype(np.uint32)


def restat_moved(s64, h, mag_orc, b64, b32, moved):
    """The oracle's in-window statistics with the moved pixels' window membership taken the GPU's way
    (only a pixel that crossed the window border changes them); values are the oracle's own."""
    s = dict(s64)
    for p in moved:
        x = mag_orc[h["band_plus"], p] - mag_orc[h["band_minus"], p]
        y = mag_orc[h["band_y"], p]
        if b64[p] >= 0 and b32[p] < 0:
            s["n_in"] -= 1; s["n_out"] += 1; s["sum_x"] -= x; s["sum_y"] -= y
        elif b64[p] < 0 and b32[p] >= 0:
            s["n_in"] += 1; s["n_out"] -= 1; s["sum_x"] += x; s["sum_y"] += y
    return s


def lnl_poisson_parity(lnl_gpu, parts, data, like_floor, label=""):
    """parts: list of (H64, b64, b32, moved) per Hess spec, data: concatenated data Hess.  Applies the 1e-4
    bar end to end (after re-binning moved edge pixels, if any) and prints what happened."""
    want_raw, want_reb, off, n_moved = 0.0, 0.0, 0, 0
    for H64, b64, b32, moved in parts:
        nb = H64.size
        d = data[off:off + nb]
        off += nb
        want_raw += O.loglike_poisson(H64, d, like_floor)
        want_reb += O.loglike_poisson(rebin_moved(H64, b64, b32, moved), d, like_floor) if moved.size else \
            O.loglike_poisson(H64, d, like_floor)
        n_moved += int(moved.size)
    if not np.isfinite(want_reb):
        assert lnl_gpu == want_reb
        return n_moved
    rel_raw = abs(lnl_gpu - want_raw) / abs(want_raw) if np.isfinite(want_raw) and want_raw != 0 else float("nan")
    rel_reb = abs(lnl_gpu - want_reb) / abs(want_reb)
    print("[lnL parity %s] moved edge pixels: %d; |dlnL|/|lnL| end to end %.3e, after re-binning them %.3e "
          "(lnL %.6f)" % (label, n_moved, rel_raw, rel_reb, lnl_gpu))
    assert rel_reb <= LNL_RTOL
    if n_moved == 0:
        assert rel_raw <= LNL_RTOL
    return n_moved
