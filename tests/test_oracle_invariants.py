"""Pins P1-P4, P8, P9 for the CPU oracle: what the paper and the mathematics fix.

P1  Eq. (6) holds on every bond after every attempt.
P2  deposition only: heights never decrease; from a flat surface the first attempt is accepted.
P3  sum h == accepted deposits, hmean == accepted / L^2, W2(t=0) == 0  (flat start).
P4  random-deposition limit (restriction can never bind): hmean(t) == t exactly and
    <W2> == t (1 - 1/L^2) for serial RS, t (1 - 1/S^2) for DT(S,K), every K  (closed form).
P8  same-colour tiles are independent: visiting them in a shuffled order, or on several threads,
    gives identical heights (the double-tiling claim of P:77).
P9  W2 of Eq. (2) recomputed from read-back heights with exact rationals.
"""
from fractions import Fraction

import numpy as np
import pytest


def literal_attempt(h, N, x, y):
    """Eq. (6) with reading Q1, written out independently of the oracle (numpy, no wrap tricks)."""
    L = h.shape[0]
    c = int(h[y, x]) + 1
    for (xx, yy) in (((x - 1) % L, y), ((x + 1) % L, y), (x, (y - 1) % L), (x, (y + 1) % L)):
        if abs(c - int(h[yy, xx])) > N:
            return 0
    h[y, x] = c
    return 1


def test_attempt_matches_literal_rule_on_random_surfaces(oracle_mod):
    rng = np.random.default_rng(5)
    for L in (2, 3, 4, 7, 8):
        for N in (1, 2, 3):
            # a valid RSOS surface: grow one with the literal rule
            h = np.zeros((L, L), dtype=np.int32)
            for _ in range(40 * L * L):
                literal_attempt(h, N, int(rng.integers(L)), int(rng.integers(L)))
            assert oracle_mod.violations(h, N) == 0
            for _ in range(200):
                x, y = int(rng.integers(L)), int(rng.integers(L))
                a, b = h.copy(), h.copy()
                ra = oracle_mod.attempt(a, N, x, y)
                rb = literal_attempt(b, N, x, y)
                assert ra == rb and (a == b).all()
                h = a


def test_violations_counter_sees_a_bad_bond(oracle_mod):
    h = np.zeros((4, 4), dtype=np.int32)
    assert oracle_mod.violations(h, 1) == 0
    h[1, 2] = 2                      # four bonds of height difference 2 > N = 1
    assert oracle_mod.violations(h, 1) == 4
    assert oracle_mod.violations(h, 2) == 0
    h[0, 0] = -3                     # wrap-around bonds are counted too
    assert oracle_mod.violations(h, 2) == 4


@pytest.mark.parametrize("L,N,R,S,K,mcs", [(32, 1, 8, 64, 1, 12), (16, 2, 4, 8, 1, 10), (64, 1, 3, 16, 4, 6),
                                           (128, 3, 2, 64, 1, 3), (64, 1, 2, 32, 32, 4), (6, 1, 5, 64, 1, 20)])
def test_invariants_every_attempt(oracle_mod, L, N, R, S, K, mcs):
    o = oracle_mod.Oracle(L, N, R, seed=11, tile=S, subsweeps=K, check_each=True)
    W2, hm = o.width()
    assert (W2 == 0).all() and (hm == 0).all()                    # P3, flat start
    prev = o.heights()
    for t in range(mcs):
        o.advance(1)
        h = o.heights()
        assert (h >= prev).all()                                   # P2
        for r in range(R):
            assert oracle_mod.violations(h[r], N) == 0             # P1 (independent full check)
        S1, S2, acc = o.sums()
        assert (S1 == acc).all()                                   # P3
        assert (S1 == h.reshape(R, -1).astype(np.int64).sum(1)).all()
        W2, hm = o.width()
        assert np.array_equal(hm, acc / float(L * L))
        # a deposit is attempted L^2 times per MCS: 0 < accepted <= L^2 * t
        assert (acc > 0).all() and (acc <= (t + 1) * L * L).all()
        prev = h
    assert o.debug_violations() == 0                               # P1 + P2 after every attempt
    assert o.t == mcs
    o.close()


def test_first_attempt_from_flat_is_accepted(oracle_mod):
    for L in (2, 5, 32):
        h = np.zeros((L, L), dtype=np.int32)
        assert oracle_mod.attempt(h, 1, L - 1, 0) == 1 and h[0, L - 1] == 1 and h.sum() == 1
        # a second deposit on the same site would make a step of 2 > N = 1
        assert oracle_mod.attempt(h, 1, L - 1, 0) == 0 and h.sum() == 1
        assert oracle_mod.attempt(h, 2, L - 1, 0) == 1 and h[0, L - 1] == 2


@pytest.mark.parametrize("L,S,K,R,tmax", [(16, 64, 1, 4096, 6), (32, 8, 1, 2048, 6), (32, 8, 2, 2048, 6),
                                          (64, 16, 2, 1024, 4), (128, 64, 1, 256, 3)])
def test_random_deposition_limit(oracle_mod, L, S, K, R, tmax):
    """P4.  N = 10^9: every attempt accepted.  Each site receives Binomial(S^2/K, 1/S^2) deposits per
    sub-sweep (tile side S; S = L in RS mode), independently across sub-sweeps, the total being fixed,
    so hmean = t exactly and E[W2] = Var(h_site) = t (1 - 1/S^2)."""
    o = oracle_mod.Oracle(L, 10 ** 9, R, seed=3, tile=S, subsweeps=K)
    Se = S if o.mode == "DT" else L
    for t in range(1, tmax + 1):
        o.advance(1)
        W2, hm = o.width()
        S1, S2, acc = o.sums()
        assert (acc == t * L * L).all() and (hm == float(t)).all()
        want = t * (1.0 - 1.0 / Se ** 2)
        se = W2.std(ddof=1) / np.sqrt(R)
        assert abs(W2.mean() - want) <= 4.0 * se, (t, W2.mean(), want, se)
        if Se <= 8:
            # resolution check: the RS and DT closed forms differ by more than the tolerance here
            assert 4.0 * se < t * (1.0 / Se ** 2 - 1.0 / (4 * Se) ** 2)
    o.close()


def test_site_draw_is_uniform(oracle_mod):
    """In the random-deposition limit h(x) counts the draws of site x: chi-square against uniform,
    per realization-summed histogram (catches a slot decoded from the wrong bits / overlapping bits)."""
    for L, S, K in ((32, 64, 1), (64, 16, 1), (64, 32, 4), (512, 64, 1)):
        R, t = (64, 40) if L < 512 else (2, 40)
        o = oracle_mod.Oracle(L, 10 ** 9, R, seed=17, tile=S, subsweeps=K)
        o.advance(t)
        h = o.heights().astype(np.int64).sum(0)
        o.close()
        mean = R * t
        chi2 = ((h - mean) ** 2).sum() / mean
        dof = L * L - 1
        # fixed totals per tile make the variance slightly smaller than Poisson: factor (1 - 1/Se^2)
        z = (chi2 - dof) / np.sqrt(2.0 * dof)
        assert abs(z) < 5.0, (L, S, K, chi2, dof, z)
        # x and y marginals (row / column sums) are uniform as well
        for ax in (0, 1):
            m = h.sum(ax)
            zz = (((m - m.mean()) ** 2).sum() / m.mean() - (L - 1)) / np.sqrt(2.0 * (L - 1))
            assert abs(zz) < 5.0


def test_16_bit_and_32_bit_slot_paths_both_used(oracle_mod):
    # S = 256 is the largest tile with 16-bit slots (2 lg S = 16); S = 512 needs 32-bit slots.
    for L, S in ((512, 256), (1024, 512)):
        o = oracle_mod.Oracle(L, 1, 1, seed=2, tile=S, check_each=True)
        assert o.mode == "DT"
        o.advance(1)
        S1, S2, acc = o.sums()
        h = o.heights()[0]
        assert oracle_mod.violations(h, 1) == 0 and o.debug_violations() == 0
        # growth velocity after 1 MCS from flat, N = 1: <hmean> = 0.652
        assert abs(acc[0] / float(L * L) - 0.652) < 0.01
        o.close()


@pytest.mark.parametrize("L,N,S,K", [(64, 1, 8, 1), (128, 2, 32, 4), (256, 1, 64, 1)])
def test_tile_order_and_thread_independence(oracle_mod, L, N, S, K):
    """P8: tiles of one colour never touch the same or adjacent sites."""
    ref = oracle_mod.Oracle(L, N, 1, seed=9, tile=S, subsweeps=K, threads=1)
    ref.advance(5)
    want = ref.heights()
    for shuffle, threads in ((1234, 1), (99, 4), (0, 8)):
        o = oracle_mod.Oracle(L, N, 1, seed=9, tile=S, subsweeps=K, threads=threads, shuffle_seed=shuffle)
        o.advance(2)
        o.advance(3)                                              # and advance() composes in time
        assert np.array_equal(o.heights(), want)
        assert np.array_equal(o.sums()[2], ref.sums()[2])
        o.close()
    ref.close()


def test_realizations_are_pure_functions_of_their_global_index(oracle_mod):
    # SURVEY 8c.1 note (iii): any subset of realizations can be run alone (first_real offset).
    a = oracle_mod.Oracle(64, 1, 6, seed=4, tile=16, subsweeps=2)
    b = oracle_mod.Oracle(64, 1, 2, seed=4, tile=16, subsweeps=2, first_real=3)
    a.advance(4)
    b.advance(4)
    assert np.array_equal(a.heights(3, 2), b.heights())
    assert not np.array_equal(a.heights(0, 1), a.heights(1, 1))
    # a different seed gives a different path
    c = oracle_mod.Oracle(64, 1, 1, seed=5, tile=16, subsweeps=2)
    c.advance(4)
    assert not np.array_equal(c.heights(), a.heights(0, 1))
    a.close(); b.close(); c.close()


def test_snapshot_restart(oracle_mod):
    a = oracle_mod.Oracle(64, 2, 3, seed=8, tile=32)
    a.advance(7)
    h7, acc7 = a.heights(), a.sums()[2]
    a.advance(2)
    b = oracle_mod.Oracle(64, 2, 3, seed=8, tile=32)
    b.set_state(h7, 7, acc7)
    b.advance(2)
    assert np.array_equal(a.heights(), b.heights()) and np.array_equal(a.sums()[2], b.sums()[2])
    a.close(); b.close()


def test_width_against_exact_rationals(oracle_mod):
    """P9: Eq. (2), W2 = <h^2> - <h>^2 over the L^2 sites, from the heights with exact rationals."""
    for L, N, S in ((32, 1, 64), (64, 3, 16), (12, 2, 64)):
        o = oracle_mod.Oracle(L, N, 3, seed=21, tile=S)
        o.advance(9)
        h = o.heights()
        W2, hm = o.width()
        S1, S2, _ = o.sums()
        for r in range(3):
            v = [int(x) for x in h[r].ravel()]
            n = L * L
            m1 = Fraction(sum(v), n)
            m2 = Fraction(sum(x * x for x in v), n)
            w = m2 - m1 * m1
            # equivalent textbook form: mean squared deviation from the mean
            assert w == sum((Fraction(x) - m1) ** 2 for x in v) / n
            assert S1[r] == sum(v) and int(S2[r]) == sum(x * x for x in v)
            assert W2[r] == float(w) or abs(W2[r] - float(w)) <= 2 ** -52 * float(w)
            assert hm[r] == float(m1)
        o.close()
    # hand example: heights 0,1,1,2 on 2x2 -> mean 1, W2 = (1+0+0+1)/4 = 1/2
    o = oracle_mod.Oracle(2, 5, 1, seed=1)
    o.set_state(np.array([[0, 1], [1, 2]], dtype=np.int32), 0)
    W2, hm = o.width()
    assert W2[0] == 0.5 and hm[0] == 1.0
    o.close()


def test_bad_arguments(oracle_mod):
    for kw in (dict(L=1, N=1, R=1), dict(L=32, N=0, R=1), dict(L=32, N=1, R=0),
               dict(L=128, N=1, R=1, tile=24), dict(L=128, N=1, R=1, tile=4),
               dict(L=128, N=1, R=1, tile=8, subsweeps=4), dict(L=128, N=1, R=1, tile=16, subsweeps=3)):
        with pytest.raises(ValueError):
            oracle_mod.Oracle(kw.pop("L"), kw.pop("N"), kw.pop("R"), 1, **kw)
