"""ctypes/numpy wrapper of the CPU oracle (oracle/pcmd_oracle.c).

TEST INFRASTRUCTURE, NOT THE PRODUCT.  Only tests/, __graft_entry__.smoke() and
bench.py's cpu_baseline / --impl reference legs may import this module.  It imports
nothing from paper_1904_00011_b200 (the CUDA path) and the CUDA path imports nothing
from here.  Workload dictionaries come from workloads/ (seeded input generators that
hold none of the method's arithmetic).

A "workload" is a dict of plain numpy arrays / scalars, see workloads/synthetic.py.
"""
from __future__ import annotations

import ctypes as C
import os
import subprocess

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "pcmd_oracle.c")
_HDR = os.path.join(_HERE, "pcmd_oracle.h")
_LIB = os.path.join(_HERE, "liboracle_pcmd.so")


def build(force: bool = False) -> str:
    """gcc -O2 -ffp-contract=off -fopenmp -shared (no -ffast-math, no -march)."""
    stale = (not os.path.exists(_LIB)) or any(
        os.path.getmtime(s) > os.path.getmtime(_LIB) for s in (_SRC, _HDR))
    if force or stale:
        cmd = ["gcc", "-O2", "-ffp-contract=off", "-fopenmp", "-shared", "-fPIC", "-std=c11",
               "-Wall", "-o", _LIB, _SRC, "-lm"]
        subprocess.run(cmd, check=True)
    return _LIB


class _Config(C.Structure):
    _fields_ = [("n_im", C.c_int32), ("n_bands", C.c_int32), ("n_age", C.c_int32),
                ("n_feh", C.c_int32), ("n_points", C.c_int32),
                ("age_idx", C.c_void_p), ("feh_idx", C.c_void_p), ("imf_w", C.c_void_p),
                ("absmag", C.c_void_p), ("feh_grid", C.c_void_p), ("zp", C.c_void_p),
                ("dust_coef", C.c_void_p), ("psf", C.c_void_p), ("psf_k", C.c_int32),
                ("sky", C.c_void_p), ("read_sigma", C.c_void_p),
                ("shot_noise", C.c_int32), ("poisson_sky", C.c_int32),
                ("dust_frac", C.c_double), ("dust_mode", C.c_int32), ("mdf_cut", C.c_double),
                ("psf_grid", C.c_int32)]


class _Params(C.Structure):
    _fields_ = [("sfh", C.c_void_p), ("feh_mean", C.c_double), ("feh_sigma", C.c_double),
                ("dmod", C.c_double), ("dust_med", C.c_double), ("dust_sigma", C.c_double)]


class _HessSpec(C.Structure):
    _fields_ = [("band_plus", C.c_int32), ("band_minus", C.c_int32), ("band_y", C.c_int32),
                ("x_lo", C.c_double), ("x_hi", C.c_double), ("y_lo", C.c_double), ("y_hi", C.c_double),
                ("nx", C.c_int32), ("ny", C.c_int32)]


class _HessStats(C.Structure):
    _fields_ = [("n_in", C.c_uint32), ("n_out", C.c_uint32), ("n_bad", C.c_uint32),
                ("sum_x", C.c_double), ("sum_y", C.c_double)]


_lib = None


def lib():
    global _lib
    if _lib is None:
        L = C.CDLL(build())
        L.orc_poisson_table.restype = C.c_int64
        L.orc_poisson_table.argtypes = [C.c_double, C.c_void_p, C.c_int64, C.POINTER(C.c_int64), C.POINTER(C.c_int64)]
        for f in (L.orc_poisson_draw, L.orc_poisson_draw_linear):
            f.restype = C.c_uint32
            f.argtypes = [C.c_void_p, C.c_int64, C.c_int64, C.c_uint32]
        L.orc_splitmix64.restype = C.c_uint64
        L.orc_splitmix64.argtypes = [C.c_uint64]
        L.orc_expneg.restype = C.c_double
        L.orc_expneg.argtypes = [C.c_double]
        L.orc_normal.restype = C.c_double
        L.orc_normal.argtypes = [C.c_uint32, C.c_uint32]
        L.orc_loglike_poisson.restype = C.c_double
        L.orc_loglike_poisson.argtypes = [C.c_void_p, C.c_void_p, C.c_int64, C.c_double]
        L.orc_loglike_gauss.restype = C.c_double
        L.orc_loglike_gauss.argtypes = [C.c_void_p, C.c_void_p, C.c_void_p, C.c_void_p, C.c_int64, C.c_int]
        L.orc_stage2.argtypes = [C.c_void_p, C.c_void_p, C.c_void_p, C.c_uint64, C.c_uint32,
                                 C.c_void_p, C.c_int64, C.c_void_p, C.c_void_p, C.c_void_p, C.c_void_p]
        L.orc_stage2_agg.argtypes = [C.c_void_p, C.c_void_p, C.c_void_p, C.c_uint64, C.c_uint32,
                                     C.c_void_p, C.c_int64, C.c_void_p, C.c_void_p, C.c_void_p, C.c_void_p, C.c_void_p]
        L.orc_stage2_brute.argtypes = [C.c_void_p, C.c_void_p, C.c_void_p, C.c_uint64, C.c_uint32,
                                       C.c_void_p, C.c_void_p]
        L.orc_stage3.argtypes = [C.c_void_p, C.c_void_p, C.c_uint64, C.c_uint32, C.c_void_p, C.c_void_p, C.c_void_p]
        L.orc_stage4.argtypes = [C.c_void_p, C.c_void_p, C.c_void_p]
        L.orc_stage5.argtypes = [C.c_void_p, C.c_uint64, C.c_uint32, C.c_void_p, C.c_void_p]
        L.orc_hess.argtypes = [C.c_void_p, C.c_int64, C.c_int32, C.c_void_p, C.c_void_p, C.c_void_p,
                               C.c_double, C.c_void_p, C.c_void_p, C.c_int64]
        L.orc_hess_f32.argtypes = [C.c_void_p, C.c_int64, C.c_int32, C.c_void_p, C.c_void_p, C.c_void_p]
        L.orc_hess_pixels.argtypes = [C.c_void_p, C.c_int64, C.c_int32, C.c_void_p, C.c_double, C.c_double,
                                      C.c_void_p, C.c_void_p]
        L.orc_hess_pixels_f32.argtypes = [C.c_void_p, C.c_int64, C.c_int32, C.c_void_p, C.c_void_p]
        L.orc_stage1.argtypes = [C.c_void_p, C.c_void_p, C.c_void_p, C.c_void_p, C.c_void_p]
        L.orc_philox4x32_10.argtypes = [C.c_void_p, C.c_void_p, C.c_void_p]
        _lib = L
    return _lib


def _p(a):
    return None if a is None else a.ctypes.data


def num_threads() -> int:
    return int(lib().orc_num_threads())


# --------------------------------------------------------------------------- primitives
def philox(key, ctr) -> np.ndarray:
    k = np.asarray(key, dtype=np.uint32)
    c = np.asarray(ctr, dtype=np.uint32)
    out = np.zeros(4, dtype=np.uint32)
    lib().orc_philox4x32_10(_p(k), _p(c), _p(out))
    return out


def splitmix64(j: int) -> int:
    return int(lib().orc_splitmix64(C.c_uint64(j)))


def expneg(t: float) -> float:
    return float(lib().orc_expneg(t))


def normal(w0: int, w1: int) -> float:
    return float(lib().orc_normal(w0, w1))


def poisson_table(lam: float):
    """Returns (T uint64[k_lo..k_hi], k_lo, k_hi)."""
    klo, khi = C.c_int64(0), C.c_int64(0)
    cap = 64
    while True:
        T = np.zeros(cap, dtype=np.uint64)
        n = lib().orc_poisson_table(lam, _p(T), cap, C.byref(klo), C.byref(khi))
        if n >= 0:
            return T[:n].copy(), int(klo.value), int(khi.value)
        if n == -1:
            raise ValueError("lambda out of range: %r" % lam)
        cap = -n - 1


def poisson_draw(T, k_lo, k_hi, u, linear=False) -> int:
    f = lib().orc_poisson_draw_linear if linear else lib().orc_poisson_draw
    return int(f(_p(T), k_lo, k_hi, int(u)))


# --------------------------------------------------------------------------- model
class Oracle:
    """Holds the marshalled config of one workload (see workloads/synthetic.py)."""

    def __init__(self, wl: dict):
        self.wl = wl
        self.N, self.B = int(wl["n_im"]), int(wl["n_bands"])
        self.J, self.A, self.Z = int(wl["n_points"]), int(wl["n_age"]), int(wl["n_feh"])
        self.P = self.N * self.N
        k = self._keep = {}
        k["age_idx"] = np.ascontiguousarray(wl["age_idx"], dtype=np.int32)
        k["feh_idx"] = np.ascontiguousarray(wl["feh_idx"], dtype=np.int32)
        for name in ("imf_w", "absmag", "feh_grid", "zp", "dust_coef", "sky", "read_sigma"):
            k[name] = np.ascontiguousarray(wl[name], dtype=np.float64)
        G = int(wl.get("psf_grid", 1) or 1)
        if G > 1:
            k["psf"] = np.ascontiguousarray(wl["psf_grid2d"], dtype=np.float64)  # [B][G*G][K][K]
            assert k["psf"].shape == (self.B, G * G, wl["psf_k"], wl["psf_k"])
        else:
            k["psf"] = np.ascontiguousarray(wl["psf2d"], dtype=np.float64)  # [B][K][K]
            assert k["psf"].shape == (self.B, wl["psf_k"], wl["psf_k"])
        assert k["absmag"].shape == (self.J, self.B)
        self.cfg = _Config(self.N, self.B, self.A, self.Z, self.J,
                           _p(k["age_idx"]), _p(k["feh_idx"]), _p(k["imf_w"]), _p(k["absmag"]),
                           _p(k["feh_grid"]), _p(k["zp"]), _p(k["dust_coef"]), _p(k["psf"]),
                           int(wl["psf_k"]), _p(k["sky"]), _p(k["read_sigma"]),
                           int(wl["shot_noise"]), int(wl["poisson_sky"]), float(wl["dust_frac"]),
                           int(wl["dust_mode"]), float(wl["mdf_cut"]), G)

    def _params(self, prm: dict):
        sfh = np.ascontiguousarray(prm["sfh"], dtype=np.float64)
        assert sfh.shape == (self.A,)
        return _Params(_p(sfh), float(prm["feh_mean"]), float(prm["feh_sigma"]), float(prm["dmod"]),
                       float(prm["dust_med"]), float(prm["dust_sigma"])), sfh

    def stage1(self, prm):
        pr, _keep = self._params(prm)
        mdfw = np.zeros(self.Z)
        lam = np.zeros(self.J)
        flux = np.zeros((self.J, self.B))
        rc = lib().orc_stage1(C.byref(self.cfg), C.byref(pr), _p(mdfw), _p(lam), _p(flux))
        if rc:
            raise ValueError("orc_stage1 failed")
        return mdfw, lam, flux

    def stage2(self, lam, flux, seed, model=0, pix=None, want_counts=False):
        if pix is None:
            n = self.P
            pixp = None
        else:
            pix = np.ascontiguousarray(pix, dtype=np.uint32)
            n, pixp = pix.size, _p(pix)
        F = np.zeros((self.B, n))
        total = np.zeros(n, dtype=np.uint32)
        h = np.zeros(n, dtype=np.uint64)
        counts = np.zeros((n, self.J), dtype=np.uint32) if want_counts else None
        lam = np.ascontiguousarray(lam, dtype=np.float64)
        flux = np.ascontiguousarray(flux, dtype=np.float64)
        rc = lib().orc_stage2(C.byref(self.cfg), _p(lam), _p(flux), C.c_uint64(seed), model, pixp, n,
                              _p(F), _p(total), _p(h), _p(counts))
        if rc:
            raise ValueError("orc_stage2 failed")
        return (F, total, h, counts) if want_counts else (F, total, h)

    def stage2_agg(self, lam, flux, seed, model=0, pix=None, want_counts=False):
        """Aggregated sampler (PAPER.md:75 fn. 3; DESIGN.md R-A1).  Returns (F, total, hash, weights[, counts])."""
        if pix is None:
            n, pixp = self.P, None
        else:
            pix = np.ascontiguousarray(pix, dtype=np.uint32)
            n, pixp = pix.size, _p(pix)
        F = np.zeros((self.B, n))
        total = np.zeros(n, dtype=np.uint32)
        h = np.zeros(n, dtype=np.uint64)
        wts = np.zeros(self.J, dtype=np.uint64)
        counts = np.zeros((n, self.J), dtype=np.uint32) if want_counts else None
        lam = np.ascontiguousarray(lam, dtype=np.float64)
        flux = np.ascontiguousarray(flux, dtype=np.float64)
        rc = lib().orc_stage2_agg(C.byref(self.cfg), _p(lam), _p(flux), C.c_uint64(seed), model, pixp, n,
                                  _p(F), _p(total), _p(h), _p(counts), _p(wts))
        if rc:
            raise ValueError("orc_stage2_agg failed")
        return (F, total, h, wts, counts) if want_counts else (F, total, h, wts)

    def stage2_brute(self, lam, flux, seed, model=0):
        F = np.zeros((self.B, self.P))
        total = np.zeros(self.P, dtype=np.uint32)
        lam = np.ascontiguousarray(lam, dtype=np.float64)
        flux = np.ascontiguousarray(flux, dtype=np.float64)
        rc = lib().orc_stage2_brute(C.byref(self.cfg), _p(lam), _p(flux), C.c_uint64(seed), model, _p(F), _p(total))
        if rc:
            raise ValueError("orc_stage2_brute failed")
        return F, total

    def stage3(self, prm, F_raw, seed, model=0):
        pr, _keep = self._params(prm)
        F_raw = np.ascontiguousarray(F_raw, dtype=np.float64)
        A = np.zeros(self.P)
        Fd = np.zeros((self.B, self.P))
        lib().orc_stage3(C.byref(self.cfg), C.byref(pr), C.c_uint64(seed), model, _p(F_raw), _p(A), _p(Fd))
        return A, Fd

    def stage4(self, F_in):
        F_in = np.ascontiguousarray(F_in, dtype=np.float64)
        G = np.zeros((self.B, self.P))
        lib().orc_stage4(C.byref(self.cfg), _p(F_in), _p(G))
        return G

    def stage5(self, G, seed, model=0):
        G = np.ascontiguousarray(G, dtype=np.float64)
        mag = np.zeros((self.B, self.P))
        rc = lib().orc_stage5(C.byref(self.cfg), C.c_uint64(seed), model, _p(G), _p(mag))
        if rc:
            raise ValueError("orc_stage5 failed")
        return mag

    def simulate(self, prm, seed, model=0):
        """Stages 1-5.  Returns a dict with every intermediate."""
        mdfw, lam, flux = self.stage1(prm)
        if int(self.wl.get("sampler_mode", 0) or 0) == 1:
            F_raw, total, h, _ = self.stage2_agg(lam, flux, seed, model)
        else:
            F_raw, total, h = self.stage2(lam, flux, seed, model)
        A, F_dust = self.stage3(prm, F_raw, seed, model)
        G = self.stage4(F_dust)
        mag = self.stage5(G, seed, model)
        return dict(mdfw=mdfw, lam=lam, flux=flux, F_raw=F_raw, total=total, hash=h, A=A,
                    F_dust=F_dust, G=G, mag=mag)

    # ---- Hess / likelihood
    @staticmethod
    def _spec(h: dict):
        return _HessSpec(int(h["band_plus"]), int(h["band_minus"]), int(h["band_y"]),
                         float(h["x_lo"]), float(h["x_hi"]), float(h["y_lo"]), float(h["y_hi"]),
                         int(h["nx"]), int(h["ny"]))

    def hess(self, h: dict, mag, edge_tol=1e-5, want_edges=False):
        mag = np.ascontiguousarray(mag, dtype=np.float64)
        n_pix = mag.shape[1]
        sp = self._spec(h)
        H = np.zeros((h["ny"], h["nx"]), dtype=np.uint32)
        st = _HessStats()
        n_edge = C.c_uint32(0)
        edges = np.zeros(n_pix if want_edges else 1, dtype=np.uint32)
        lib().orc_hess(C.byref(sp), n_pix, mag.shape[0], _p(mag), _p(H), C.byref(st), edge_tol,
                       C.byref(n_edge), _p(edges) if want_edges else None, edges.size)
        stats = dict(n_in=st.n_in, n_out=st.n_out, n_bad=st.n_bad, sum_x=st.sum_x, sum_y=st.sum_y,
                     n_edge=int(n_edge.value))
        if want_edges:
            stats["edges"] = edges[: n_edge.value].copy()
        return H, stats

    def hess_f32(self, h: dict, mag32):
        mag32 = np.ascontiguousarray(mag32, dtype=np.float32)
        n_pix = mag32.shape[1]
        sp = self._spec(h)
        H = np.zeros((h["ny"], h["nx"]), dtype=np.uint32)
        st = _HessStats()
        lib().orc_hess_f32(C.byref(sp), n_pix, mag32.shape[0], _p(mag32), _p(H), C.byref(st))
        return H, dict(n_in=st.n_in, n_out=st.n_out, n_bad=st.n_bad, sum_x=st.sum_x, sum_y=st.sum_y)


    def hess_pixels(self, h: dict, mag, tol_x=2e-5, tol_y=1e-5):
        """Per-pixel bin index of the fp64 Hess (-1 outside, -2 NaN) and the near-edge flags
        (bit 0: colour within tol_x of an edge, bit 1: magnitude within tol_y)."""
        mag = np.ascontiguousarray(mag, dtype=np.float64)
        n_pix = mag.shape[1]
        sp = self._spec(h)
        b = np.zeros(n_pix, dtype=np.int32)
        near = np.zeros(n_pix, dtype=np.uint8)
        lib().orc_hess_pixels(C.byref(sp), n_pix, mag.shape[0], _p(mag), tol_x, tol_y, _p(b), _p(near))
        return b, near

    def hess_pixels_f32(self, h: dict, mag32):
        """Per-pixel bin index of the kernel-precision Hess decision (orc_hess_f32)."""
        mag32 = np.ascontiguousarray(mag32, dtype=np.float32)
        n_pix = mag32.shape[1]
        sp = self._spec(h)
        b = np.zeros(n_pix, dtype=np.int32)
        lib().orc_hess_pixels_f32(C.byref(sp), n_pix, mag32.shape[0], _p(mag32), _p(b))
        return b


def _stats_struct(s: dict):
    return _HessStats(int(s["n_in"]), int(s["n_out"]), int(s["n_bad"]), float(s["sum_x"]), float(s["sum_y"]))


def loglike_poisson(hess_model, hess_data, m_floor=0.1) -> float:
    hm = np.ascontiguousarray(hess_model, dtype=np.uint32).ravel()
    hd = np.ascontiguousarray(hess_data, dtype=np.uint32).ravel()
    assert hm.size == hd.size
    return float(lib().orc_loglike_poisson(_p(hm), _p(hd), hm.size, m_floor))


def loglike_gauss(hess_model, stats_model, hess_data, stats_data, literal=False) -> float:
    hm = np.ascontiguousarray(hess_model, dtype=np.uint32).ravel()
    hd = np.ascontiguousarray(hess_data, dtype=np.uint32).ravel()
    sm, sd = _stats_struct(stats_model), _stats_struct(stats_data)
    return float(lib().orc_loglike_gauss(_p(hm), C.byref(sm), _p(hd), C.byref(sd), hm.size, int(literal)))
