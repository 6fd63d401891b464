"""Pin P5: the oracle's serial RS dynamics against an exact Markov-chain enumeration
of the RSOS rule (Eq. (6)) on 2x2, 3x3 and 4x4 periodic lattices.

The enumeration below is a brute force over all site sequences (weights = number of sequences
reaching a configuration) written from the rule alone; it shares nothing with the oracle.  It is
first checked against tests/golden/markov_small_lattice.txt, then the oracle's ensemble means over
many realizations must agree with the exact expectations within 4 standard errors.
"""
import os
from fractions import Fraction

import numpy as np
import pytest

HERE = os.path.dirname(os.path.abspath(__file__))


def enumerate_rsos(L, N, kmax):
    """Exact E[W2], E[hmean] after k = 1..kmax uniformly random deposition attempts, flat start."""
    n = L * L
    nb = [[y * L + (x - 1) % L, y * L + (x + 1) % L, ((y - 1) % L) * L + x, ((y + 1) % L) * L + x]
          for y in range(L) for x in range(L)]
    dist = {(0,) * n: 1}
    out = {}
    for k in range(1, kmax + 1):
        new = {}
        for s, w in dist.items():
            for i in range(n):
                c = s[i] + 1
                ok = True
                for j in nb[i]:
                    if abs(c - s[j]) > N:
                        ok = False
                        break
                s2 = s[:i] + (c,) + s[i + 1:] if ok else s
                new[s2] = new.get(s2, 0) + w
        dist = new
        num_w = 0
        num_h = 0
        for s, w in dist.items():
            s1 = sum(s)
            sq = sum(v * v for v in s)
            num_w += w * (n * sq - s1 * s1)
            num_h += w * s1
        tot = n ** k
        out[k] = (Fraction(num_w, n * n * tot), Fraction(num_h, n * tot))
    return out


def golden_rows():
    rows = []
    for l in open(os.path.join(HERE, "golden", "markov_small_lattice.txt")):
        if not l.strip() or l[0] == "#":
            continue
        L, N, k, w_ex, w_dec, h_ex, h_dec = l.split()
        rows.append((int(L), int(N), int(k), w_ex, float(w_dec), h_ex, float(h_dec)))
    return rows


_ENUM_CACHE = {}


def exact(L, N, kmax):
    key = (L, N)
    if key not in _ENUM_CACHE or max(_ENUM_CACHE[key]) < kmax:
        _ENUM_CACHE[key] = enumerate_rsos(L, N, kmax)
    return _ENUM_CACHE[key]


@pytest.mark.parametrize("L,N,kmax", [(2, 1, 16), (2, 2, 16), (3, 1, 18), (3, 2, 18), (4, 1, 16)])
def test_golden_file_matches_enumeration(L, N, kmax):
    ex = exact(L, N, kmax)
    n_checked = 0
    for (gL, gN, k, w_ex, w_dec, h_ex, h_dec) in golden_rows():
        if (gL, gN) != (L, N):
            continue
        w, h = ex[k]
        if w_ex != "-":
            assert Fraction(w_ex) == w
        if h_ex != "-":
            assert Fraction(h_ex) == h
        assert abs(float(w) - w_dec) < 1e-9
        assert abs(float(h) - h_dec) < 1e-9
        n_checked += 1
    assert n_checked >= 1


def test_random_deposition_row_of_the_table():
    # last row of the P5 table: N >= k  =>  E[W2] = (k/L^2)(1 - 1/L^2), E[hmean] = k/L^2
    for L, k in [(2, 6), (3, 5)]:
        w, h = enumerate_rsos(L, 10 ** 6, k)[k]
        n = L * L
        assert w == Fraction(k, n) * (1 - Fraction(1, n))
        assert h == Fraction(k, n)


@pytest.mark.parametrize("L,N,R,tmax", [(2, 1, 1 << 20, 4), (2, 2, 1 << 20, 4), (3, 1, 1 << 18, 2),
                                        (3, 2, 1 << 18, 2), (4, 1, 1 << 18, 1)])
def test_oracle_ensemble_matches_enumeration(oracle_mod, L, N, R, tmax):
    n = L * L
    ex = exact(L, N, n * tmax)
    o = oracle_mod.Oracle(L, N, R, seed=20160509 + 7 * L + N)
    assert o.mode == "RS"
    for t in range(1, tmax + 1):
        o.advance(1)
        W2, hm = o.width()
        w_ex, h_ex = ex[n * t]
        for got, want, name in ((W2, float(w_ex), "W2"), (hm, float(h_ex), "hmean")):
            se = got.std(ddof=1) / np.sqrt(R)
            assert abs(got.mean() - want) <= 4.0 * se, (name, L, N, t, got.mean(), want, se)
            # and the test has teeth: the tolerance is far below the effect of, e.g., one neighbour dropped
            assert 4.0 * se < 0.01 * max(want, 0.05)
    o.close()
