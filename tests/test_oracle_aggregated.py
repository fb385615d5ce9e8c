"""Pins of the oracle's aggregated sampler (PAPER.md:75 footnote 3; DESIGN.md R-A1): brute force in Python
integers on tiny images, closed-form moments, the Poisson total, degenerate cases."""
import numpy as np

from oracle import pcmd_oracle as O
from workloads import synthetic as W


def _brute(lam, seed, model, P):
    """Independent restatement with Python integers: returns (counts [P][J], weights)."""
    J = lam.size
    Lam = 0.0
    for x in lam:
        Lam += float(x)
    w = [int((float(x) / Lam) * 2.0 ** 40 + 0.5) for x in lam]
    C = [0]
    for x in w:
        C.append(C[-1] + x)
    T, k_lo, k_hi = O.poisson_table(Lam)
    key = (seed & 0xFFFFFFFF, seed >> 32)
    counts = np.zeros((P, J), dtype=np.int64)
    for p in range(P):
        N = O.poisson_draw(T, k_lo, k_hi, int(O.philox(key, (p, 0, model, 4))[0]), linear=True)
        for s in range(N):
            ws = O.philox(key, (p, 1 + s // 2, model, 4))
            U = (int(ws[2 * (s % 2)]) << 32) | int(ws[2 * (s % 2) + 1])
            r = (U * C[-1]) >> 64
            j = max(i for i in range(J) if C[i] <= r)          # the definition: C_j <= r < C_{j+1}
            assert r < C[j + 1]
            counts[p, j] += 1
    return counts, np.array(w, dtype=np.uint64)


def test_aggregated_sampler_matches_python_integer_brute_force():
    for J, seed, model in ((8, 5, 0), (13, (7 << 32) | 9, 3)):
        wl = W.tiny_model(n_im=4, J=J)
        orc = O.Oracle(wl)
        _, lam, flux = orc.stage1(wl["params"][0])
        F, total, h, wts, counts = orc.stage2_agg(lam, flux, seed, model, want_counts=True)
        want, w = _brute(lam, seed, model, 16)
        assert np.array_equal(wts, w)
        assert np.array_equal(counts, want) and np.array_equal(total, want.sum(1))
        assert np.allclose(F, (want @ flux).T, rtol=1e-12)
        mult = np.array([O.splitmix64(j) | 1 for j in range(J)], dtype=object)
        assert [int(x) for x in h] == [int(sum(int(n) * m for n, m in zip(row, mult)) % 2 ** 64) for row in want]


def test_aggregated_sampler_moments_and_total():
    wl = W.scaled(W.config(1), 96)
    orc = O.Oracle(wl)
    _, lam, flux = orc.stage1(wl["params"][0])
    F, total, _, wts, counts = orc.stage2_agg(lam, flux, seed=11, want_counts=True)
    P, Lam = total.size, lam.sum()
    # the pixel total is Poisson(N_pix) (PAPER.md:75 fn. 3): mean = variance = N_pix
    assert abs(total.mean() - Lam) < 5 * np.sqrt(Lam / P)
    assert abs(total.var() / Lam - 1.0) < 5 * np.sqrt(2.0 / P)
    # compound Poisson closed forms (north_star): E[F_b] = sum lambda f, Var[F_b] = sum lambda f^2
    mean, var = lam @ flux, lam @ flux ** 2
    assert np.all(np.abs(F.mean(1) - mean) < 5 * np.sqrt(var / P))
    # every point's count is Poisson(lambda_j) marginally
    z = (counts.sum(0) - P * lam) / np.sqrt(P * lam)
    assert np.all(np.abs(z[lam * P > 50]) < 5.5) and abs(z[lam * P > 50].std() - 1.0) < 0.2
    # integer weights: lambda_j / N_pix to 2^-40 each
    assert np.max(np.abs(wts.astype(np.float64) / 2.0 ** 40 - lam / Lam)) <= 2.0 ** -40
    assert abs(int(wts.sum()) - 2 ** 40) <= lam.size


def test_aggregated_sampler_degenerate_cases():
    wl = W.tiny_model(n_im=4, J=8)
    orc = O.Oracle(wl)
    _, lam, flux = orc.stage1(wl["params"][0])
    F, total, h, _ = orc.stage2_agg(np.zeros_like(lam), flux, seed=1)
    assert not F.any() and not total.any() and not h.any()
    one = np.zeros_like(lam)
    one[3] = 6.5                                   # a single populated point: every star is that point
    F, total, h, wts, counts = orc.stage2_agg(one, flux, seed=1, want_counts=True)
    assert np.array_equal(counts[:, 3], total) and counts.sum() == total.sum() and total.sum() > 0
    assert np.allclose(F, np.outer(flux[3], total), rtol=1e-13)
    # a pixel subset gives the same pixels
    sub = np.array([5, 2, 15], dtype=np.uint32)
    Fs, ts, hs, _ = orc.stage2_agg(lam, flux, seed=4, pix=sub)
    Ff, tf, hf, _ = orc.stage2_agg(lam, flux, seed=4)
    assert np.array_equal(Fs, Ff[:, sub]) and np.array_equal(ts, tf[sub]) and np.array_equal(hs, hf[sub])
