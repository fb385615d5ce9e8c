"""Seeded synthetic inputs shaped like the paper's workloads.

This module serves BOTH the CPU oracle and the CUDA path and therefore holds none of
the method's arithmetic: it only manufactures input tables (isochrones, PSFs, filter
constants, parameter draws) with numpy and reads the frozen constants under
workloads/frozen/ (written once by oracle/freeze_workloads.py, which calls only the
oracle).  It imports neither oracle/ nor paper_1904_00011_b200/.

The paper's workloads use MIST isochrones, Tiny Tim PSFs and ACS filter data
(PAPER.md:137,178-180); none are available offline, so the tables below stand in for
them, keeping their shapes and value structure: hundreds of points per isochrone
(PAPER.md:194), tens of isochrones, a steep IMF so
most points are faint and numerous and a few bright and rare, 2-3 bands,
N_im 64-1024.

The five configurations are BASELINE.json's `configs` c1..c5.
"""
from __future__ import annotations

import json
import os

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
FROZEN_DIR = os.path.join(_HERE, "frozen")

ZP = 26.0 + 2.5 * np.log10(3000.0)          # ACS-like zero-point + exposure
FEH_GRID5 = np.array([-1.0, -0.75, -0.5, -0.25, 0.0])   # 0.25 dex grid
_A = np.array([5.4, 5.1, 4.8])              # bluest -> reddest
_BETA_LO = np.array([4.8, 4.4, 4.0])
_BETA_HI = np.array([3.4, 3.2, 3.0])
_GAMMA = np.array([0.4, 0.25, 0.1])
N_GIANT = 20


def _isochrone(log_age: float, feh: float, K: int, bands):
    """One synthetic isochrone: K points (K-20 main sequence + 20 giants).
    Returns imf_w[K] (sum 1) and absmag[K][len(bands)]."""
    m_to = float(np.clip((10.0 ** log_age / 1e10) ** (-0.4), 0.5, 100.0))
    n_ms = K - N_GIANT
    m_ms = np.exp(np.linspace(np.log(0.1), np.log(m_to), n_ms))
    m_g = m_to * (1.0 + 0.02 * (np.arange(N_GIANT) + 1.0) / N_GIANT)
    m = np.concatenate([m_ms, m_g])
    # power-law IMF (slope -2.3) integrated over cells bounded by geometric mid-points
    e = np.empty(K + 1)
    e[1:-1] = np.sqrt(m[:-1] * m[1:])
    e[0] = m[0] * m[0] / e[1]
    e[-1] = m[-1] * m[-1] / e[-2]
    w = (e[:-1] ** (-1.3) - e[1:] ** (-1.3)) / 1.3
    w = w / w.sum()
    # main sequence: broken power-law mass-magnitude relation, metallicity term
    lm = np.log10(m_ms)[:, None]
    beta = np.where(m_ms[:, None] <= 1.0, _BETA_LO[None, :], _BETA_HI[None, :])
    M_ms = _A[None, :] - 2.5 * beta * lm + _GAMMA[None, :] * feh
    # giants: reddest band linear from the turn-off to the tip, colours redden with s
    s = ((np.arange(N_GIANT) + 1.0) / N_GIANT)[:, None]
    to = M_ms[-1]
    tip = -4.0 - 1.5 * np.log10(m_to)
    red = to[2] + (tip - to[2]) * s[:, 0]
    dcol = (1.2 + 0.5 * feh) * s[:, 0]
    M_g = np.empty((N_GIANT, 3))
    M_g[:, 2] = red
    M_g[:, 0] = red + (to[0] - to[2]) + dcol
    M_g[:, 1] = red + (to[1] - to[2]) + 0.5 * dcol
    M = np.concatenate([M_ms, M_g], axis=0)
    return w, M[:, list(bands)]


def _grid(log_ages, fehs, K, bands):
    age_idx, feh_idx, imf_w, absmag = [], [], [], []
    for a, t in enumerate(log_ages):
        for z, f in enumerate(fehs):
            w, M = _isochrone(float(t), float(f), K, bands)
            age_idx.append(np.full(K, a, dtype=np.int32))
            feh_idx.append(np.full(K, z, dtype=np.int32))
            imf_w.append(w)
            absmag.append(M)
    return (np.concatenate(age_idx), np.concatenate(feh_idx), np.concatenate(imf_w),
            np.concatenate(absmag, axis=0))


def gaussian_psf_factor(K: int, sigma: float) -> np.ndarray:
    """1-D factor a[K] (fp32, sum ~ 1) of the separable Gaussian PSF a (x) a; the 2-D
    sampled Gaussian exp(-(dx^2+dy^2)/2 sigma^2) normalised to 1 IS this outer product."""
    r = (K - 1) // 2
    d = np.arange(-r, r + 1, dtype=np.float64)
    g = np.exp(-0.5 * (d / sigma) ** 2)
    return (g / g.sum()).astype(np.float32)


def _psfs(B, K, sigmas):
    f = np.stack([gaussian_psf_factor(K, s) for s in sigmas])          # [B][K] fp32
    f64 = f.astype(np.float64)
    p2 = np.einsum("bi,bj->bij", f64, f64)                               # exact products
    return f, p2


def _frozen(name: str, allow_unfrozen: bool):
    path = os.path.join(FROZEN_DIR, name + ".json")
    if os.path.exists(path):
        with open(path) as fh:
            return json.load(fh)
    if allow_unfrozen:
        return None
    raise FileNotFoundError(path + " missing: run `python oracle/freeze_workloads.py`")


def _hess(bp, bm, by, x_lo, x_hi, y_lo, y_hi, nx, ny):
    return dict(band_plus=bp, band_minus=bm, band_y=by, x_lo=float(x_lo), x_hi=float(x_hi),
                y_lo=float(y_lo), y_hi=float(y_hi), nx=int(nx), ny=int(ny))


def dense_hess(sparse: dict, ny: int, nx: int) -> np.ndarray:
    H = np.zeros(ny * nx, dtype=np.uint32)
    H[np.asarray(sparse["idx"], dtype=np.int64)] = np.asarray(sparse["cnt"], dtype=np.uint32)
    return H.reshape(ny, nx)


def sparse_hess(H: np.ndarray) -> dict:
    flat = np.asarray(H).ravel()
    idx = np.nonzero(flat)[0]
    return dict(idx=[int(i) for i in idx], cnt=[int(c) for c in flat[idx]])


def _base(name, n_im, bands, log_ages, fehs, K, psf_k, psf_sigmas):
    B = len(bands)
    age_idx, feh_idx, imf_w, absmag = _grid(log_ages, fehs, K, bands)
    psf1d, psf2d = _psfs(B, psf_k, psf_sigmas)
    return dict(
        name=name, n_im=int(n_im), n_bands=B, n_age=len(log_ages), n_feh=len(fehs),
        n_points=int(age_idx.size), age_idx=age_idx, feh_idx=feh_idx, imf_w=imf_w, absmag=absmag,
        log_ages=np.asarray(log_ages, dtype=np.float64), feh_grid=np.asarray(fehs, dtype=np.float64),
        zp=np.full(B, ZP), dust_coef=np.zeros(B), psf_k=int(psf_k), psf1d=psf1d, psf2d=psf2d,
        sky=np.zeros(B), read_sigma=np.zeros(B), shot_noise=1, poisson_sky=0,
        dust_frac=0.5, dust_mode=0, mdf_cut=0.01, like_floor=0.1, seed=0, data_seed=1,
    )


def _attach_frozen(wl, fz, default_hess):
    """Hess windows / data Hess / read noise frozen by oracle/freeze_workloads.py."""
    if fz is None:
        wl["hess"] = default_hess
        wl["data_hess"] = None
        wl["data_stats"] = None
        wl["frozen"] = False
        return wl
    wl["hess"] = fz["hess"]
    wl["data_hess"] = [dense_hess(s, h["ny"], h["nx"]) for s, h in zip(fz["data_hess"], fz["hess"])]
    wl["data_stats"] = fz["data_stats"]
    if "read_sigma" in fz:
        wl["read_sigma"] = np.asarray(fz["read_sigma"], dtype=np.float64)
    wl["frozen"] = True
    return wl


def config(c: int, allow_unfrozen: bool = False) -> dict:
    """BASELINE.json configs[c-1] as a workload dict: tables + `params` (list of models)."""
    rng = np.random.default_rng(20190400 + c)
    if c == 1:
        wl = _base("c1", 64, (0, 2), [10.0], [0.0], 256, 5, [1.0, 1.0])
        wl["shot_noise"] = 0
        wl["params"] = [dict(sfh=np.array([100.0]), feh_mean=0.0, feh_sigma=0.2, dmod=24.0,
                             dust_med=0.0, dust_sigma=0.0)]
        fz = _frozen("c1", allow_unfrozen)
        # BASELINE c1: 64x64 bins over colour [-1,3] and mag [-6,6] read relative to dmod (R-Q13)
        wl = _attach_frozen(wl, fz, [_hess(0, 1, 1, -1.0, 3.0, 18.0, 30.0, 64, 64)])
        if fz is not None:
            wl["hess"] = [_hess(0, 1, 1, -1.0, 3.0, 18.0, 30.0, 64, 64)]
        return wl
    ages7 = np.linspace(6.6, 10.2, 7)
    if c == 2:
        wl = _base("c2", 256, (0, 2), ages7, FEH_GRID5, 300, 7, [1.0, 1.0])
        wl["params"] = [dict(sfh=1e3 * rng.dirichlet(np.ones(7)), feh_mean=-0.5, feh_sigma=0.2,
                             dmod=27.0, dust_med=0.0, dust_sigma=0.0)]
        return _attach_frozen(wl, _frozen("c2", allow_unfrozen),
                              [_hess(0, 1, 1, -2.0, 3.0, 18.0, 30.0, 100, 100)])
    if c == 3:
        wl = _base("c3", 512, (0, 1, 2), ages7, FEH_GRID5, 300, 15, [1.0, 1.2, 1.5])
        wl["dust_coef"] = np.array([1.2, 1.0, 0.6])
        wl["dust_mode"] = 1
        wl["dust_frac"] = 0.5
        wl["sky"] = np.full(3, 100.0)
        wl["read_sigma"] = np.full(3, 5.0)
        wl["poisson_sky"] = 1
        wl["params"] = [dict(sfh=1e4 * rng.dirichlet(np.ones(7)), feh_mean=-0.5, feh_sigma=0.2,
                             dmod=29.5, dust_med=0.5, dust_sigma=0.2)]
        return _attach_frozen(wl, _frozen("c3", allow_unfrozen),
                              [_hess(0, 2, 2, -2.0, 3.0, 18.0, 30.0, 100, 100),
                               _hess(1, 2, 2, -2.0, 3.0, 18.0, 30.0, 100, 100)])
    if c == 4:
        wl = _base("c4", 256, (0, 2), ages7, FEH_GRID5, 300, 7, [1.0, 1.0])
        wl["dust_coef"] = np.array([1.2, 0.6])
        wl["dust_mode"] = 1
        wl["dust_frac"] = 0.5
        prm = []
        for _ in range(64):
            prm.append(dict(sfh=1e3 * rng.dirichlet(np.ones(7)), feh_mean=float(rng.uniform(-1.5, 0.3)),
                            feh_sigma=float(rng.uniform(0.05, 0.5)), dmod=float(rng.uniform(25.0, 31.0)),
                            dust_med=float(rng.uniform(0.0, 1.0)), dust_sigma=0.2))
        wl["params"] = prm
        # c4 is c2 batched: one fixed data Hess, c2's (R-Q16)
        return _attach_frozen(wl, _frozen("c2", allow_unfrozen),
                              [_hess(0, 1, 1, -2.0, 3.0, 18.0, 30.0, 100, 100)])
    if c == 5:
        ages10 = np.linspace(6.6, 10.2, 10)
        wl = _base("c5", 1024, (0, 2), ages10, FEH_GRID5, 400, 21, [2.0, 2.0])
        wl["params"] = [dict(sfh=np.full(10, 1e5), feh_mean=-0.5, feh_sigma=0.2, dmod=35.0,
                             dust_med=0.0, dust_sigma=0.0)]
        return _attach_frozen(wl, _frozen("c5", allow_unfrozen),
                              [_hess(0, 1, 1, -2.0, 3.0, 18.0, 30.0, 200, 200)])
    raise ValueError("config must be 1..5")


def scaled(wl: dict, n_im: int, name: str | None = None) -> dict:
    """Same tables on a smaller (or larger) image: the parity-test sizes."""
    out = dict(wl)
    out["n_im"] = int(n_im)
    out["name"] = name or "%s@%d" % (wl["name"], n_im)
    return out


def with_psf(wl: dict, psf_k: int, sigmas) -> dict:
    out = dict(wl)
    out["psf_k"] = int(psf_k)
    out["psf1d"], out["psf2d"] = _psfs(wl["n_bands"], psf_k, sigmas)
    return out


def with_psf_grid(wl: dict, G: int = 4) -> dict:
    """Sub-pixel PSF grid: G x G Gaussian PSFs per band, the one of cell (gy, gx) shifted
    by ((gx + 0.5) / G - 0.5, (gy + 0.5) / G - 0.5) pixel, each normalised to 1 (fp32)."""
    out = dict(wl)
    K, B = int(wl["psf_k"]), int(wl["n_bands"])
    r = (K - 1) // 2
    d = np.arange(-r, r + 1, dtype=np.float64)
    # recover each band's sigma from its 1-D factor: ratio of the two central samples
    grid = np.empty((B, G * G, K, K), dtype=np.float32)
    for b in range(B):
        f = wl["psf1d"][b].astype(np.float64)
        sigma = 1.0 if K < 3 else float(np.sqrt(0.5 / np.log(f[r] / f[r + 1])))
        for gy in range(G):
            for gx in range(G):
                sx, sy = (gx + 0.5) / G - 0.5, (gy + 0.5) / G - 0.5
                p = np.exp(-0.5 * (((d[None, :] - sx) / sigma) ** 2 + ((d[:, None] - sy) / sigma) ** 2))
                grid[b, gy * G + gx] = (p / p.sum()).astype(np.float32)
    out["psf_grid"] = int(G)
    out["psf_grid2d"] = grid
    out["name"] = wl["name"] + "+grid%d" % G
    return out


def tiny_model(n_im=4, J=8, B=2, seed=7, lam_scale=1.0) -> dict:
    """A 4x4-image, J-point, single-isochrone workload for brute-force checks."""
    rng = np.random.default_rng(seed)
    wl = _base("tiny", n_im, (0, 2)[:B] if B <= 2 else (0, 1, 2), [10.0], [0.0], max(J, N_GIANT + 2), 3,
               [0.8] * B)
    # keep only J points, re-normalise the IMF weights
    sel = np.sort(rng.choice(wl["n_points"], size=J, replace=False))
    for k in ("age_idx", "feh_idx", "imf_w", "absmag"):
        wl[k] = wl[k][sel]
    wl["imf_w"] = wl["imf_w"] / wl["imf_w"].sum()
    wl["n_points"] = J
    wl["params"] = [dict(sfh=np.array([20.0 * lam_scale]), feh_mean=0.0, feh_sigma=0.2, dmod=20.0,
                         dust_med=0.0, dust_sigma=0.0)]
    wl["hess"] = [_hess(0, 1, 1, -1.0, 3.0, 10.0, 30.0, 16, 16)]
    wl["data_hess"] = None
    wl["data_stats"] = None
    wl["frozen"] = False
    return wl
