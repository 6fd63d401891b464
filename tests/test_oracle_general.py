"""Pins for the general-L schedule RSG / DTG (S 8(f) NEXT-3: the paper's L = 9605, and
its irregular tilings "a subset of domains have larger lateral size"): lattice sides that are not powers of two.

  * the bounded draw is EXACTLY uniform: census over all 2^32 words -- every value is hit floor(2^32 / n) times and
    2^32 mod n words are rejected (the mathematics of multiply-shift with rejection);
  * the tiles partition the lattice (edges floor(i L / T)), widths differ by at most one and lie in [S, 2S);
  * P1-P3 (Eq. 6 after every attempt, monotone heights, sum h = accepted) on general lattices;
  * P4: random-deposition limit: hmean = t exactly, <W^2> = t (1 - T^2 / L^2) for DTG (each of the T^2 tiles of n
    sites gives every site Binomial(n, 1/n) hits per MCS) and t (1 - 1/L^2) for RSG -- closed forms;
  * DTG agrees with serial RSG statistically (coarse band, like P7).
The 3x3 Markov-chain pin (tests/test_oracle_markov.py) runs through RSG as well.
"""
import numpy as np
import pytest


@pytest.mark.parametrize("n", [3, 4160, 9605])
def test_bounded_draw_census_is_exactly_uniform(oracle_mod, n):
    counts, rejected = oracle_mod.bounded_census(n)
    assert rejected == (1 << 32) % n
    assert (counts == (1 << 32) // n).all()


def test_bounded_draw_by_hand(oracle_mod):
    # n = 3: thr = 2^32 mod 3 = 1; v = 0: m = 0, low word 0 < 1 -> rejected; v = 1: m = 3, low 3 >= 1, value 0;
    # v = 0x55555556: m = 0x1_0000_0002 -> value 1; v = 0xFFFFFFFF: m = 0x2_FFFF_FFFD -> value 2
    assert oracle_mod.bounded(0, 3) == (0, False)
    assert oracle_mod.bounded(1, 3) == (0, True)
    assert oracle_mod.bounded(0x55555556, 3) == (1, True)
    assert oracle_mod.bounded(0xFFFFFFFF, 3) == (2, True)
    # a power of two never rejects and takes the top bits
    assert oracle_mod.bounded(0xABCDEF01, 256) == (0xAB, True)


@pytest.mark.parametrize("L,S", [(150, 64), (200, 32), (9605, 64), (191, 64), (100, 8)])
def test_tiles_partition_the_lattice(L, S):
    T = 2 * (L // (2 * S))
    edges = [(i * L) // T for i in range(T + 1)]
    assert edges[0] == 0 and edges[-1] == L and T % 2 == 0
    w = np.diff(edges)
    assert w.min() >= S and w.max() < 2 * S and w.max() - w.min() <= 1 and w.sum() == L


@pytest.mark.parametrize("L,N,R,S,K,mcs", [(150, 1, 3, 64, 1, 6), (200, 2, 2, 32, 4, 4), (100, 1, 2, 8, 2, 5),
                                           (6, 1, 4, 64, 1, 30), (45, 3, 2, 64, 1, 10)])
def test_invariants_every_attempt_general(oracle_mod, L, N, R, S, K, mcs):
    o = oracle_mod.Oracle(L, N, R, seed=4, tile=S, subsweeps=K, check_each=True)
    assert o.mode == ("DT" if 2 * S <= L else "RS")
    prev = o.heights()
    for _ in range(mcs):
        o.advance(1)
        h = o.heights()
        assert (h >= prev).all()
        prev = h
    assert o.debug_violations() == 0
    S1, S2, acc = o.sums()
    assert (S1 == acc).all() and (acc > 0).all() and (acc <= mcs * L * L).all()
    for r in range(R):
        assert oracle_mod.violations(h[r], N) == 0
    o.close()


@pytest.mark.parametrize("L,S,K", [(150, 64, 1), (200, 32, 4), (96, 8, 1), (45, 64, 1)])
def test_random_deposition_limit_general(oracle_mod, L, S, K):
    R, t = 96, 6
    o = oracle_mod.Oracle(L, 10 ** 9, R, seed=8, tile=S, subsweeps=K)
    o.advance(t)
    W2, hm = o.width()
    assert (hm == t).all()                                   # every attempt accepted, L^2 attempts per MCS
    T = 2 * (L // (2 * S)) if 2 * S <= L else 1
    expect = t * (1.0 - T * T / float(L * L))
    se = W2.std(ddof=1) / np.sqrt(R)
    assert abs(W2.mean() - expect) < 4 * se, (W2.mean(), expect, se)
    o.close()


def test_dtg_vs_serial_coarse_band(oracle_mod):
    """L = 150: DTG(64, K) (T = 2: four tiles of 75 x 75) against serial RSG, N = 1, 512 realizations, t = 10.
    A coarse regression band, like P7: the decomposition bias at S ~ 64 is a few 10^-3."""
    L, R, t = 150, 512, 10
    ref = oracle_mod.Oracle(L, 1, R, seed=21, tile=128)
    assert ref.mode == "RS"
    ref.advance(t)
    w_ref, h_ref = ref.width()
    ref.close()
    for K in (1, 4):
        o = oracle_mod.Oracle(L, 1, R, seed=22 + K, tile=64, subsweeps=K)
        assert o.mode == "DT"
        o.advance(t)
        w, h = o.width()
        o.close()
        d = w.mean() / w_ref.mean() - 1.0
        assert -0.012 < d < 0.008, (K, d)
        assert abs(h.mean() / h_ref.mean() - 1.0) < 0.004
