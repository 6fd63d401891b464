"""Pins for the oracle's moment functions (Eq. 13-15).

rsos_oracle_height_moments is Eq. (13) with the empirical height distribution of one surface; it is
pinned by hand-worked examples (values derived in the comments below, not by the oracle), by scipy's
independent moment / skew / kurtosis routines, and by the exact integer power sums through the
binomial expansion in python big integers / fractions.
"""
from fractions import Fraction

import numpy as np
import pytest


def _with_heights(oracle_mod, h):
    h = np.asarray(h, dtype=np.int32)
    L = h.shape[-1]
    o = oracle_mod.Oracle(L, 10 ** 9, 1, seed=1, tile=2 * L)          # RS mode, any L >= 2
    o.set_state(h.reshape(1, L, L), 0)
    return o


def test_hand_worked_2x2_examples(oracle_mod):
    # heights {0,1,1,2}: mean 1, deviations -1,0,0,1 -> Phi2 = 2/4, Phi3 = 0, Phi4 = 2/4; S = 0, Q = 0.5/0.25 - 3 = -1
    o = _with_heights(oracle_mod, [[0, 1], [1, 2]])
    hb, (p2, p3, p4) = o.height_moments(0)
    assert hb == 1.0 and (p2, p3, p4) == (0.5, 0.0, 0.5)
    assert p4 / p2 ** 2 - 3 == -1.0
    o.close()
    # heights {0,0,0,4}: mean 1, deviations -1,-1,-1,3 -> Phi2 = 12/4 = 3, Phi3 = 24/4 = 6, Phi4 = 84/4 = 21
    o = _with_heights(oracle_mod, [[0, 0], [0, 4]])
    hb, (p2, p3, p4) = o.height_moments(0)
    assert hb == 1.0 and (p2, p3, p4) == (3.0, 6.0, 21.0)
    assert abs(p3 / p2 ** 1.5 - 2 / np.sqrt(3)) < 1e-15              # skewness 6 / 3^(3/2) = 2/sqrt(3)
    assert abs((p4 / p2 ** 2 - 3) - (21 / 9 - 3)) < 1e-15            # excess kurtosis -2/3
    o.close()
    # a non-integer mean: {0,0,0,1}: mean 1/4, deviations -1/4 (x3), 3/4 -> Phi2 = 3/16, Phi3 = 3/32, Phi4 = 21/256
    o = _with_heights(oracle_mod, [[0, 0], [0, 1]])
    hb, (p2, p3, p4) = o.height_moments(0)
    assert (hb, p2, p3, p4) == (0.25, 3 / 16, 3 / 32, 21 / 256)
    # power sums about base 0 and base -2, by hand: M_k(0) = 1 for all k; M_k(-2): 3 * 2^k + 3^k
    assert o.power_sums(0, 0) == [1, 1, 1, 1]
    assert o.power_sums(0, -2) == [3 * 2 + 3, 3 * 4 + 9, 3 * 8 + 27, 3 * 16 + 81]
    o.close()


def test_against_scipy_and_exact_rationals(oracle_mod):
    stats = pytest.importorskip("scipy.stats")
    rng = np.random.default_rng(7)
    for L, lo, hi in [(4, -3, 3), (16, 100000, 100040), (32, -2 ** 20, -2 ** 20 + 9)]:
        h = rng.integers(lo, hi + 1, size=(L, L)).astype(np.int32)
        o = _with_heights(oracle_mod, h)
        hb, phi = o.height_moments(0)
        x = h.ravel().astype(np.float64)
        for k, v in zip((2, 3, 4), phi):
            ref = stats.moment(x, k)                                  # library routine: k-th central moment
            assert abs(v - ref) <= 1e-9 * max(1.0, abs(ref)), (L, k, v, ref)
        assert abs(phi[1] / phi[0] ** 1.5 - stats.skew(x)) < 1e-9
        assert abs(phi[2] / phi[0] ** 2 - 3 - stats.kurtosis(x)) < 1e-9
        # exact: central moments from the integer power sums by the binomial theorem, in rationals
        n = L * L
        xs = [int(v) for v in h.ravel()]
        base = sum(xs) // n
        M = o.power_sums(0, base)
        assert M == [sum((v - base) ** k for v in xs) for k in (1, 2, 3, 4)]
        m1 = Fraction(M[0], n)
        mu2 = Fraction(M[1], n) - m1 ** 2
        mu3 = Fraction(M[2], n) - 3 * m1 * Fraction(M[1], n) + 2 * m1 ** 3
        mu4 = Fraction(M[3], n) - 4 * m1 * Fraction(M[2], n) + 6 * m1 ** 2 * Fraction(M[1], n) - 3 * m1 ** 4
        for v, ex in zip(phi, (mu2, mu3, mu4)):
            assert abs(v - float(ex)) <= 1e-12 * max(1.0, abs(float(ex)))
        assert abs(hb - float(Fraction(sum(xs), n))) <= 1e-15 * max(1.0, abs(hb))
        o.close()


def test_flat_and_shifted_surfaces(oracle_mod):
    """Invariants: a flat surface has all central moments 0; adding a constant changes none of them;
    mirroring h -> -h flips the sign of the odd one only."""
    rng = np.random.default_rng(11)
    o = _with_heights(oracle_mod, np.full((8, 8), 17))
    assert o.height_moments(0) == (17.0, [0.0, 0.0, 0.0])
    o.close()
    h = rng.integers(0, 12, size=(8, 8))
    a = _with_heights(oracle_mod, h).height_moments(0)
    b = _with_heights(oracle_mod, h + 1000).height_moments(0)
    c = _with_heights(oracle_mod, -h).height_moments(0)
    assert np.allclose(a[1], b[1], rtol=1e-13, atol=0)
    assert np.allclose([a[1][0], -a[1][1], a[1][2]], c[1], rtol=1e-13, atol=0)
