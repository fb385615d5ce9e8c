"""ctypes binding of libpcmd.so (include/pcmd.h): argument marshalling only.

PyTorch is used for device buffers and streams, nothing else.  Every method maps 1:1 onto the
C entry point of the same name; every step of the path runs in the CUDA kernels.
"""
from __future__ import annotations

import ctypes as C
import os
import re

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_LIB_PATH = os.environ.get("PCMD_LIBRARY") or os.path.join(_HERE, "libpcmd.so")   # PCMD_LIBRARY: an alternative build
_HEADER = os.path.join(os.path.dirname(_HERE), "include", "pcmd.h")

LIKE_POISSON, LIKE_GAUSS, LIKE_GAUSS_LITERAL = 0, 1, 2
MAX_BANDS, MAX_HESS = 4, 4


class PcmdError(RuntimeError):
    def __init__(self, code, what=""):
        self.code = code
        msg = lib().pcmd_strerror(code).decode() if _lib is not None else str(code)
        super().__init__("%s: %s (code %d)" % (what, msg, code))


class HessSpec(C.Structure):
    _fields_ = [("band_plus", C.c_int32), ("band_minus", C.c_int32), ("band_y", C.c_int32),
                ("x_lo", C.c_double), ("x_hi", C.c_double), ("y_lo", C.c_double), ("y_hi", C.c_double),
                ("nx", C.c_int32), ("ny", C.c_int32)]


class HessStats(C.Structure):
    _fields_ = [("n_in", C.c_uint32), ("n_out", C.c_uint32), ("n_bad", C.c_uint32), ("_pad", C.c_uint32),
                ("sum_x", C.c_double), ("sum_y", C.c_double)]


STATS_DTYPE = np.dtype([("n_in", "<u4"), ("n_out", "<u4"), ("n_bad", "<u4"), ("_pad", "<u4"),
                        ("sum_x", "<f8"), ("sum_y", "<f8")])


class Config(C.Structure):
    _fields_ = [("n_im", C.c_int32), ("n_bands", C.c_int32), ("n_age", C.c_int32), ("n_feh", C.c_int32),
                ("n_points", C.c_int32),
                ("age_idx", C.c_void_p), ("feh_idx", C.c_void_p), ("imf_w", C.c_void_p),
                ("absmag", C.c_void_p), ("feh_grid", C.c_void_p), ("zp", C.c_void_p),
                ("dust_coef", C.c_void_p), ("psf", C.c_void_p), ("psf_k", C.c_int32),
                ("psf_separable", C.c_int32), ("sky", C.c_void_p), ("read_sigma", C.c_void_p),
                ("shot_noise", C.c_int32), ("poisson_sky", C.c_int32), ("like_floor", C.c_double),
                ("n_hess", C.c_int32), ("hess", C.c_void_p), ("dust_frac", C.c_double),
                ("dust_mode", C.c_int32), ("mdf_cut", C.c_double), ("psf_grid", C.c_int32),
                ("sampler_mode", C.c_int32)]


class Params(C.Structure):
    _fields_ = [("sfh", C.c_void_p), ("feh_mean", C.c_double), ("feh_sigma", C.c_double),
                ("dmod", C.c_double), ("dust_med", C.c_double), ("dust_sigma", C.c_double)]


_lib = None


def lib():
    """Loads libpcmd.so; fails loudly if it has not been built (no fallback)."""
    global _lib
    if _lib is None:
        if not os.path.exists(_LIB_PATH):
            raise ImportError("libpcmd.so is missing: run `python -m paper_1904_00011_b200.build` "
                              "(there is no CPU fallback)")
        L = C.CDLL(_LIB_PATH)
        vp, i32, i64, u64, u32 = C.c_void_p, C.c_int32, C.c_int64, C.c_uint64, C.c_uint32
        L.pcmd_strerror.restype = C.c_char_p
        L.pcmd_strerror.argtypes = [C.c_int]
        L.pcmd_create.argtypes = [C.POINTER(vp), C.POINTER(Config)]
        L.pcmd_destroy.argtypes = [vp]
        L.pcmd_destroy.restype = None
        L.pcmd_simulate.argtypes = [vp, vp, i32, u64, u32, vp, vp, vp, vp, vp]
        L.pcmd_simulate_repeat.argtypes = [vp, vp, i32, u64, u32, vp, vp, vp, vp, vp]
        L.pcmd_hess.argtypes = [vp, vp, i32, vp, vp, vp]
        L.pcmd_hess_noalloc.argtypes = [vp, vp, i32, vp, vp, vp]
        L.pcmd_hess_noalloc_setup.argtypes = []
        L.pcmd_hess_noalloc_parts.argtypes = [vp, i32]
        L.pcmd_hess_noalloc_parts.restype = i64
        L.pcmd_loglike.argtypes = [vp, vp, vp, i32, vp, vp, i32, vp, vp]
        L.pcmd_evaluate_host.argtypes = [vp, vp, i32, u64, u32, vp, vp, i32, vp, vp, vp, vp]
        L.pcmd_hess_bins_total.argtypes = [vp]
        L.pcmd_hess_bins_total.restype = i64
        L.pcmd_debug_weights.argtypes = [vp, i32, vp, vp, vp, vp, vp, i64, C.POINTER(i64)]
        L.pcmd_debug_taps.argtypes = [vp, vp, vp]
        L.pcmd_debug_philox.argtypes = [u64, vp, i64, vp]
        L.pcmd_status.argtypes = [vp, vp]
        L.pcmd_last_cuda_error.argtypes = [vp]
        L.pcmd_params_from_paper.argtypes = [i32, vp, C.c_double, C.c_double, C.c_double, C.c_double, C.c_double,
                                             vp, C.POINTER(Params)]
        L.pcmd_pipe_bench.argtypes = [i32, i32, i32, i32, vp]
        L.pcmd_pipe_bench_name.argtypes = [i32]
        L.pcmd_pipe_bench_name.restype = C.c_char_p
        L.pcmd_launch_count.argtypes = [vp]
        L.pcmd_launch_count.restype = i64
        L.pcmd_profile.argtypes = [vp, i32]
        L.pcmd_stage_ms.argtypes = [vp, vp]
        _lib = L
    return _lib


def exported_symbols():
    """Names of the functions include/pcmd.h declares (for the symbol test)."""
    with open(_HEADER) as fh:
        text = fh.read()
    return sorted(set(re.findall(r"\b(pcmd_[a-z_0-9]+)\s*\(", text)))


def _np(a):
    return None if a is None else a.ctypes.data


def _dp(t):
    return None if t is None else t.data_ptr()


def params_from_paper(log10_sfh, feh, sigma_feh, log10_ebv, sigma_dust, dmod) -> dict:
    """pcmd_params_from_paper (Table 1 free parameters -> linear fields): a params dict as the workloads use."""
    ls = np.ascontiguousarray(log10_sfh, dtype=np.float64)
    sfh = np.zeros_like(ls)
    out = Params()
    rc = lib().pcmd_params_from_paper(ls.size, _np(ls), float(feh), float(sigma_feh), float(log10_ebv),
                                      float(sigma_dust), float(dmod), _np(sfh), C.byref(out))
    if rc:
        raise PcmdError(rc, "pcmd_params_from_paper")
    return dict(sfh=sfh, feh_mean=out.feh_mean, feh_sigma=out.feh_sigma, dmod=out.dmod,
                dust_med=out.dust_med, dust_sigma=out.dust_sigma)


def pipe_bench(ctas_per_sm: int = 2, threads: int = 512, iters: int = 4096, only: str | None = None):
    """pcmd_pipe_bench for every test (or the one named `only`): list of dicts {name, rate, cycles, ms, steps_per_s}."""
    out = []
    t = 0
    while True:
        name = lib().pcmd_pipe_bench_name(t)
        if name is None:
            return out
        if only is not None and name.decode() != only:
            t += 1
            continue
        r = np.zeros(4)
        rc = lib().pcmd_pipe_bench(t, ctas_per_sm, threads, iters, _np(r))
        if rc:
            raise PcmdError(rc, "pcmd_pipe_bench")
        out.append(dict(name=name.decode(), rate=float(r[0]), cycles=float(r[1]), ms=float(r[2]),
                        steps_per_s=float(r[3])))
        t += 1


def philox(seed: int, ctr) -> np.ndarray:
    """Device Philox4x32-10 words for counters ctr[n][4] (parity of the random stream)."""
    ctr = np.ascontiguousarray(ctr, dtype=np.uint32).reshape(-1, 4)
    out = np.zeros_like(ctr)
    rc = lib().pcmd_debug_philox(C.c_uint64(seed), _np(ctr), ctr.shape[0], _np(out))
    if rc:
        raise PcmdError(rc, "pcmd_debug_philox")
    return out


class Pcmd:
    """One pcmd_ctx built from a workload dict (see workloads/synthetic.py for the keys)."""

    def __init__(self, wl: dict, separable: bool = False):
        import torch
        if not torch.cuda.is_available():
            raise RuntimeError("paper_1904_00011_b200 needs a CUDA device (no CPU fallback)")
        self.torch = torch
        self.N, self.B = int(wl["n_im"]), int(wl["n_bands"])
        self.J, self.A, self.Z = int(wl["n_points"]), int(wl["n_age"]), int(wl["n_feh"])
        self.P = self.N * self.N
        self.hess_specs = list(wl.get("hess") or [])
        k = self._keep = {}
        k["age_idx"] = np.ascontiguousarray(wl["age_idx"], dtype=np.int32)
        k["feh_idx"] = np.ascontiguousarray(wl["feh_idx"], dtype=np.int32)
        for name in ("imf_w", "absmag", "feh_grid", "zp", "dust_coef", "sky", "read_sigma"):
            k[name] = np.ascontiguousarray(wl[name], dtype=np.float64)
        K = int(wl["psf_k"])
        G = int(wl.get("psf_grid", 1) or 1)
        if G > 1:
            if separable:
                raise ValueError("a PSF grid needs psf_separable=0")
            k["psf"] = np.ascontiguousarray(wl["psf_grid2d"], dtype=np.float32)   # [B][G*G][K][K]
        elif separable:
            f = np.ascontiguousarray(wl["psf1d"], dtype=np.float32)          # [B][K]
            k["psf"] = np.ascontiguousarray(np.stack([f, f], axis=1))        # [B][2][K]
        else:
            k["psf"] = np.ascontiguousarray(wl["psf2d"], dtype=np.float32)   # [B][K][K]
        hs = (HessSpec * max(1, len(self.hess_specs)))()
        for i, h in enumerate(self.hess_specs):
            hs[i] = HessSpec(int(h["band_plus"]), int(h["band_minus"]), int(h["band_y"]), float(h["x_lo"]),
                             float(h["x_hi"]), float(h["y_lo"]), float(h["y_hi"]), int(h["nx"]), int(h["ny"]))
        k["hess"] = hs
        cfg = Config(self.N, self.B, self.A, self.Z, self.J, _np(k["age_idx"]), _np(k["feh_idx"]),
                     _np(k["imf_w"]), _np(k["absmag"]), _np(k["feh_grid"]), _np(k["zp"]), _np(k["dust_coef"]),
                     _np(k["psf"]), K, int(bool(separable)), _np(k["sky"]), _np(k["read_sigma"]),
                     int(wl["shot_noise"]), int(wl["poisson_sky"]), float(wl.get("like_floor", 0.1)),
                     len(self.hess_specs), C.addressof(hs), float(wl["dust_frac"]), int(wl["dust_mode"]),
                     float(wl["mdf_cut"]), G, int(wl.get("sampler_mode", 0) or 0))
        self._ctx = C.c_void_p()
        rc = lib().pcmd_create(C.byref(self._ctx), C.byref(cfg))
        if rc:
            raise PcmdError(rc, "pcmd_create")
        self.bins_total = int(lib().pcmd_hess_bins_total(self._ctx))

    def close(self):
        if getattr(self, "_ctx", None):
            lib().pcmd_destroy(self._ctx)
            self._ctx = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    # ---- marshalling helpers
    def _params(self, prms):
        arr = (Params * len(prms))()
        keep = []
        for i, p in enumerate(prms):
            sfh = np.ascontiguousarray(p["sfh"], dtype=np.float64)
            assert sfh.shape == (self.A,)
            keep.append(sfh)
            arr[i] = Params(_np(sfh), float(p["feh_mean"]), float(p["feh_sigma"]), float(p["dmod"]),
                            float(p["dust_med"]), float(p["dust_sigma"]))
        return arr, keep

    def _stream(self):
        return C.c_void_p(self.torch.cuda.current_stream().cuda_stream)

    # ---- entry points
    def simulate(self, prms, seed=0, model_index0=0, want_raw=False, want_counts=False, mag=None):
        t = self.torch
        n = len(prms)
        arr, keep = self._params(prms)
        if mag is None:
            mag = t.empty((n, self.B, self.N, self.N), dtype=t.float32, device="cuda")
        raw = t.empty_like(mag) if want_raw else None
        hsh = t.empty((n, self.P), dtype=t.int64, device="cuda") if want_counts else None
        tot = t.empty((n, self.P), dtype=t.int32, device="cuda") if want_counts else None
        rc = lib().pcmd_simulate(self._ctx, C.addressof(arr), n, C.c_uint64(seed), model_index0, _dp(mag),
                                 _dp(raw), _dp(hsh), _dp(tot), self._stream())
        if rc:
            raise PcmdError(rc, "pcmd_simulate")
        out = dict(mag=mag)
        if want_raw:
            out["flux_raw"] = raw
        if want_counts:
            out["hash"], out["total"] = hsh, tot
        return out

    def simulate_repeat(self, prm, n_repeats, seed=0, model_index0=0, want_raw=False, want_counts=False, mag=None):
        """n_repeats realisations of one parameter vector (stage 1 once)."""
        t = self.torch
        arr, keep = self._params([prm])
        if mag is None:
            mag = t.empty((n_repeats, self.B, self.N, self.N), dtype=t.float32, device="cuda")
        raw = t.empty_like(mag) if want_raw else None
        hsh = t.empty((n_repeats, self.P), dtype=t.int64, device="cuda") if want_counts else None
        tot = t.empty((n_repeats, self.P), dtype=t.int32, device="cuda") if want_counts else None
        rc = lib().pcmd_simulate_repeat(self._ctx, C.addressof(arr), n_repeats, C.c_uint64(seed), model_index0,
                                        _dp(mag), _dp(raw), _dp(hsh), _dp(tot), self._stream())
        if rc:
            raise PcmdError(rc, "pcmd_simulate_repeat")
        out = dict(mag=mag)
        if want_raw:
            out["flux_raw"] = raw
        if want_counts:
            out["hash"], out["total"] = hsh, tot
        return out

    def hess(self, mag, want_stats=True, out=None):
        t = self.torch
        n = mag.shape[0]
        H = out if out is not None else t.empty((n, self.bins_total), dtype=t.int32, device="cuda")
        st = t.empty((n, len(self.hess_specs), 4), dtype=t.float64, device="cuda") if want_stats else None
        rc = lib().pcmd_hess(self._ctx, _dp(mag), n, _dp(H), _dp(st), self._stream())
        if rc:
            raise PcmdError(rc, "pcmd_hess")
        return H, st

    def hess_noalloc(self, mag, out, stats=None):
        """pcmd_hess_noalloc: stage 6 into the caller's `out` (and `stats`), no allocation anywhere on the way
        (include/pcmd.h: fixed scratch of PCMD_HESS_NOALLOC_MAX_PARTS partials, shared per device)."""
        rc = lib().pcmd_hess_noalloc(self._ctx, _dp(mag), mag.shape[0], _dp(out), _dp(stats), self._stream())
        if rc:
            raise PcmdError(rc, "pcmd_hess_noalloc")
        return out, stats

    def hess_noalloc_parts(self, n_models):
        return int(lib().pcmd_hess_noalloc_parts(self._ctx, int(n_models)))

    def loglike(self, H, stats, data_hess, data_stats=None, mode=LIKE_POISSON):
        t = self.torch
        n = H.shape[0]
        out = t.empty((n,), dtype=t.float64, device="cuda")
        rc = lib().pcmd_loglike(self._ctx, _dp(H), _dp(stats), n, _dp(data_hess), _dp(data_stats), mode,
                                _dp(out), self._stream())
        if rc:
            raise PcmdError(rc, "pcmd_loglike")
        return out

    def evaluate_host(self, prms, data_hess, seed=0, model_index0=0, data_stats=None, mode=LIKE_POISSON,
                      want_hess=True):
        """HOST in / HOST out: numpy data Hess -> (lnL[n], hess[n][bins] or None, stats or None)."""
        n = len(prms)
        arr, keep = self._params(prms)
        dh = np.ascontiguousarray(data_hess, dtype=np.uint32).ravel()
        assert dh.size == self.bins_total
        ds = None if data_stats is None else np.ascontiguousarray(data_stats, dtype=STATS_DTYPE)
        lnl = np.zeros(n, dtype=np.float64)
        H = np.zeros((n, self.bins_total), dtype=np.uint32) if want_hess else None
        st = np.zeros((n, len(self.hess_specs)), dtype=STATS_DTYPE) if want_hess else None
        rc = lib().pcmd_evaluate_host(self._ctx, C.addressof(arr), n, C.c_uint64(seed), model_index0, _np(dh),
                                      _np(ds), mode, _np(lnl), _np(H), _np(st), self._stream())
        if rc:
            raise PcmdError(rc, "pcmd_evaluate_host")
        return lnl, H, st

    def debug_weights(self, model=0):
        lam = np.zeros(self.J)
        flux = np.zeros((self.J, self.B), dtype=np.float32)
        k0 = np.zeros(self.J, dtype=np.uint32)
        ln = np.zeros(self.J, dtype=np.uint32)
        n = C.c_int64(0)
        rc = lib().pcmd_debug_weights(self._ctx, model, _np(lam), _np(flux), _np(k0), _np(ln), None, 0, C.byref(n))
        if rc:
            raise PcmdError(rc, "pcmd_debug_weights")
        tab = np.zeros(max(1, n.value), dtype=np.uint32)
        rc = lib().pcmd_debug_weights(self._ctx, model, None, None, None, None, _np(tab), tab.size, C.byref(n))
        if rc:
            raise PcmdError(rc, "pcmd_debug_weights")
        return dict(lam=lam, flux=flux, k0=k0, len=ln, tables=tab[: n.value])

    def debug_taps(self, flux_dust=None, flux_conv=None):
        self._taps = (flux_dust, flux_conv)
        rc = lib().pcmd_debug_taps(self._ctx, _dp(flux_dust), _dp(flux_conv))
        if rc:
            raise PcmdError(rc, "pcmd_debug_taps")

    def status(self):
        return int(lib().pcmd_status(self._ctx, self._stream()))

    def profile(self, enable=True):
        rc = lib().pcmd_profile(self._ctx, int(bool(enable)))
        if rc:
            raise PcmdError(rc, "pcmd_profile")

    def stage_ms(self):
        """Milliseconds of stages (1, 2, 4-5, 6, 7) of the last profiled calls (synchronises)."""
        ms = np.zeros(5, dtype=np.float32)
        rc = lib().pcmd_stage_ms(self._ctx, _np(ms))
        if rc:
            raise PcmdError(rc, "pcmd_stage_ms")
        return ms

    def launch_count(self):
        return int(lib().pcmd_launch_count(self._ctx))

    @staticmethod
    def stats_to_numpy(st):
        """Device stats tensor [n][n_hess][4 x f64-sized words] -> structured numpy array."""
        return st.cpu().numpy().view(STATS_DTYPE).reshape(st.shape[0], st.shape[1])
