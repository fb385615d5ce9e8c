"""Writes workloads/frozen/c{1,2,3,5}.json: constants that the workload recipe defines
through one oracle run:

* c1 `read_sigma` = 1 % of the per-band median of the PSF-convolved image of seed 0
  (BASELINE.json c1 "Gaussian read noise at 1% of the median flux", reading R-Q12);
* Hess windows of c2/c3/c5: 0.1 %-99.9 % range of each axis of the data realisation,
  padded by 0.25 mag, rounded outward to 0.05 mag (reading R-Q13); c1's window is
  BASELINE's fixed one;
* the data Hess of every config (data seed 1, produced by the oracle) and its stats.

Calls only oracle/ and workloads/.  Usage: python oracle/freeze_workloads.py [1 2 3 5]
"""
from __future__ import annotations

import json
import math
import os
import sys
import time

import numpy as np

sys.path.insert(0, os.path.dirname(os.path.dirname(os.path.abspath(__file__))))

from oracle import pcmd_oracle as O          # noqa: E402
from workloads import synthetic as W         # noqa: E402


def _window(v):
    v = v[np.isfinite(v)]
    lo, hi = np.quantile(v, [0.001, 0.999])
    lo = math.floor((lo - 0.25) / 0.05 + 1e-9) * 0.05
    hi = math.ceil((hi + 0.25) / 0.05 - 1e-9) * 0.05
    return round(lo, 2), round(hi, 2)


def freeze(c: int):
    t0 = time.time()
    wl = W.config(c, allow_unfrozen=True)
    out = {}
    prm = wl["params"][0]
    if c == 1:
        o = O.Oracle(wl)
        _, lam, flux = o.stage1(prm)
        F, _, _ = o.stage2(lam, flux, seed=wl["seed"])
        _, Fd = o.stage3(prm, F, seed=wl["seed"])
        G = o.stage4(Fd)
        wl["read_sigma"] = 0.01 * np.median(G, axis=1)
        out["read_sigma"] = [float(x) for x in wl["read_sigma"]]
    o = O.Oracle(wl)
    sim = o.simulate(prm, seed=wl["data_seed"])
    mag = sim["mag"]
    hess = []
    for h in wl["hess"]:
        h = dict(h)
        if c != 1:
            h["x_lo"], h["x_hi"] = _window(mag[h["band_plus"]] - mag[h["band_minus"]])
            h["y_lo"], h["y_hi"] = _window(mag[h["band_y"]])
        hess.append(h)
    out["hess"] = hess
    out["data_hess"], out["data_stats"] = [], []
    for h in hess:
        H, st = o.hess(h, mag)
        out["data_hess"].append(W.sparse_hess(H))
        out["data_stats"].append({k: (int(v) if k.startswith("n_") else float(v)) for k, v in st.items()})
    out["how"] = "python oracle/freeze_workloads.py %d  (oracle only; data seed %d)" % (c, wl["data_seed"])
    os.makedirs(W.FROZEN_DIR, exist_ok=True)
    with open(os.path.join(W.FROZEN_DIR, "c%d.json" % c), "w") as fh:
        json.dump(out, fh, separators=(",", ":"))
    print("c%d frozen in %.1f s: %s" % (c, time.time() - t0,
                                        [(h["x_lo"], h["x_hi"], h["y_lo"], h["y_hi"]) for h in hess]), flush=True)
    print("   stats", out["data_stats"], flush=True)


if __name__ == "__main__":
    for c in [int(a) for a in sys.argv[1:]] or [1, 2, 3, 5]:
        freeze(c)
