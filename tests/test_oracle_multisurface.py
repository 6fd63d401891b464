"""Pins for the shared-coordinate multisurface schedule MS (S 8(f) NEXT-4).

  * P1-P3 on every attempt;
  * random-deposition limit (closed forms): a surface makes Binomial(2 L^2, 1/2) attempts per MCS (mean L^2, variance
    L^2 / 2) and <W^2> = t (1 - 1/L^2), the serial value;
  * the coordinates really are shared inside a group of 128 and only there: in the random-deposition limit two
    surfaces of one group have site-wise height correlation Var(c) / (E[c] + Var(c)) = (1 - p) / (2 - p), p = 1/L^2
    (c = number of selections of a site, Binomial(2 L^2 t, p); each surface takes each selection with an independent
    fair bit), surfaces of different groups 0;
  * with the restriction active (N = 1) the ensemble W^2(t) agrees with serial RS (coarse band): the half-update
    mask "breaks the correlation" well enough for ensemble averages.
"""
import numpy as np
import pytest


def test_invariants_every_attempt_ms(oracle_mod):
    o = oracle_mod.Oracle(16, 1, 6, seed=2, multisurface=True, check_each=True, first_real=125)   # spans two groups
    o.advance(8)
    assert o.debug_violations() == 0
    S1, _, acc = o.sums()
    assert (S1 == acc).all() and (acc > 0).all()
    for h in o.heights():
        assert oracle_mod.violations(h, 1) == 0
    o.close()


def test_random_deposition_limit_ms(oracle_mod):
    L, G, t = 16, 40, 8                                        # 40 groups of 128: surfaces of a group share their
    R = 128 * G                                                # coordinate histogram, so GROUPS are the independent samples
    o = oracle_mod.Oracle(L, 10 ** 9, R, seed=4, multisurface=True)
    o.advance(t)
    W2, hm = o.width()
    _, _, acc = o.sums()
    h = o.heights().reshape(R, -1).astype(np.float64)
    o.close()
    n = L * L
    # attempts per surface: Binomial(2 n t, 1/2), independent bits
    assert abs(acc.mean() - n * t) < 4 * np.sqrt(n * t / 2.0 / R)
    assert abs(acc.var(ddof=1) / (n * t / 2.0) - 1.0) < 0.1
    gw = W2.reshape(G, 128).mean(axis=1)
    assert abs(gw.mean() - t * (1 - 1.0 / n)) < 4 * gw.std(ddof=1) / np.sqrt(G), (gw.mean(), gw.std(ddof=1))
    # site-wise correlation between surfaces: inside a group vs across groups
    d = h - t                                                   # E[h(x)] = t
    def corr(a, b):
        return float((d[a] * d[b]).mean() / np.sqrt((d[a] ** 2).mean() * (d[b] ** 2).mean()))
    same = np.mean([corr(128 * g + i, 128 * g + i + 1) for g in range(G) for i in range(0, 126, 8)])
    cross = np.mean([corr(128 * g + i, 128 * (g + 1) + i) for g in range(G - 1) for i in range(0, 126, 8)])
    p = 1.0 / n
    assert abs(same - (1 - p) / (2 - p)) < 0.02, same
    assert abs(cross) < 0.02, cross


def test_ms_agrees_with_serial_ensemble(oracle_mod):
    L, R, t = 32, 2048, 10                                    # 16 groups
    ref = oracle_mod.Oracle(L, 1, R, seed=31)
    ref.advance(t)
    w0, h0 = ref.width()
    ref.close()
    o = oracle_mod.Oracle(L, 1, R, seed=32, multisurface=True)
    o.advance(t)
    w, h = o.width()
    o.close()
    # surfaces of a group are correlated (fewer effective samples): the standard error comes from the group means
    gw = w.reshape(-1, 128).mean(axis=1)
    se = np.hypot(gw.std(ddof=1) / np.sqrt(len(gw)), w0.std(ddof=1) / np.sqrt(R))
    assert abs(w.mean() - w0.mean()) < 4 * se and se / w0.mean() < 0.01, (w.mean(), w0.mean(), se)
    assert abs(h.mean() / h0.mean() - 1.0) < 0.01
