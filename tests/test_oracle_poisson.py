"""Pins for the Poisson variant DTP(c) of the decomposition (S 8(f) NEXT-1, SURVEY 8(c).4:
"several passes per MCS with fresh origin and Poisson attempt counts" is the variant of small domains that agrees
with serial dynamics).

  * the inversion table is floor(2^32 P(X <= k)), X ~ Poisson(4), recomputed here with 60-digit decimals;
  * counts drawn from Philox words have the Poisson(4) distribution (mean, variance, chi-square);
  * random-deposition limit: by Poisson thinning every site gets Poisson(1) attempts per MCS independently, so
    <W^2> = t (1 - 1/L^2) -- the serial value, not DT's t (1 - 1/c^2) -- and hmean fluctuates with variance t / L^2;
  * P1-P3 on every attempt; DTP(8) agrees with serial RS where DT(8,1) is off by -3.6 % (has teeth).
"""
from decimal import Decimal, getcontext

import numpy as np
import pytest


def _table():
    getcontext().prec = 60
    lam, cdf = Decimal(4), Decimal(0)
    term = (-lam).exp()
    out = []
    for k in range(23):
        cdf += term
        out.append(int((cdf * (1 << 32)).to_integral_value(rounding="ROUND_FLOOR")))
        term = term * lam / (k + 1)
    return out


def test_inversion_table_is_the_poisson_cdf(oracle_mod):
    T = _table()
    assert T[0] == 78665070 and T[22] == (1 << 32) - 1          # floor(2^32 e^-4); the tail below 2^-32 is cut
    prev = 0
    for k, tk in enumerate(T):
        if tk > prev:
            assert oracle_mod.poisson4(tk - 1) == k               # w < T[k]  <=>  n <= k
        assert oracle_mod.poisson4(tk) == k + 1
        prev = tk
    assert oracle_mod.poisson4(0) == 0 and oracle_mod.poisson4(0xFFFFFFFF) == 23


def test_counts_are_poisson_distributed(oracle_mod):
    from scipy import stats
    n = 200000
    words = [int(oracle_mod.philox((i, 7, 3, 1), (5, 0))[0]) for i in range(0, n // 50)]   # real generator words ...
    rng = np.random.default_rng(1)
    words += [int(w) for w in rng.integers(0, 1 << 32, size=n - len(words), dtype=np.uint64)]  # ... and uniform ones
    c = np.array([oracle_mod.poisson4(w) for w in words])
    assert abs(c.mean() - 4.0) < 4 * 2.0 / np.sqrt(n)
    assert abs(c.var() - 4.0) < 0.06
    obs = np.bincount(c, minlength=16)[:16].astype(float)
    obs[15] += (c >= 16).sum()
    exp = stats.poisson.pmf(np.arange(16), 4.0) * n
    exp[15] = n - exp[:15].sum()
    chi2 = ((obs - exp) ** 2 / exp).sum()
    assert chi2 < stats.chi2.ppf(0.9999, 15)


def test_random_deposition_limit_is_the_serial_one(oracle_mod):
    L, R, t = 64, 256, 6
    o = oracle_mod.Oracle(L, 10 ** 9, R, seed=3, tile=8, poisson=True)
    o.advance(t)
    W2, hm = o.width()
    o.close()
    se = W2.std(ddof=1) / np.sqrt(R)
    assert abs(W2.mean() - t * (1 - 1.0 / L ** 2)) < 4 * se
    assert abs(W2.mean() - t * (1 - 1.0 / 64)) > 6 * se          # not the fixed-count value of DT(8, K)
    assert len(set(hm.tolist())) > R // 2                          # attempt counts are random: hmean is not exactly t
    assert abs(hm.mean() - t) < 4 * np.sqrt(t / L ** 2 / R)
    assert abs(hm.var(ddof=1) / (t / L ** 2) - 1.0) < 0.4


@pytest.mark.parametrize("L,N,S", [(32, 1, 8), (64, 2, 16)])
def test_invariants_every_attempt_poisson(oracle_mod, L, N, S):
    o = oracle_mod.Oracle(L, N, 3, seed=5, tile=S, poisson=True, check_each=True)
    o.advance(6)
    assert o.debug_violations() == 0
    S1, _, acc = o.sums()
    assert (S1 == acc).all()
    for h in o.heights():
        assert oracle_mod.violations(h, N) == 0
    o.close()


def test_poisson_variant_agrees_with_serial_where_fixed_counts_do_not(oracle_mod):
    """L = 64, N = 1, 1024 realizations, t = 10: serial RS vs DTP(8) vs DT(8,1).  SE of <W^2> is about 0.1 %."""
    L, R, t = 64, 1024, 10
    res = {}
    for name, kw in (("rs", dict(tile=64)), ("dtp", dict(tile=8, poisson=True)), ("dt", dict(tile=8))):
        o = oracle_mod.Oracle(L, 1, R, seed=17 + len(name), **kw)
        o.advance(t)
        res[name] = o.width()[0]
        o.close()
    rs = res["rs"].mean()
    se = np.sqrt(res["rs"].var(ddof=1) / R + res["dtp"].var(ddof=1) / R)
    assert abs(res["dtp"].mean() - rs) < 3.5 * se, (res["dtp"].mean(), rs, se)
    assert res["dt"].mean() / rs - 1.0 < -0.02
