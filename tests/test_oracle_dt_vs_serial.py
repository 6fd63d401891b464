"""Pin P7: the domain-decomposed schedule DT(S,K) reproduces serial random-sequential
W2(t) within statistical error (BASELINE.json north_star; "match perfectly those ...
obtained by sequential Monte Carlo updates", P:204-208 domain-size study).

Serial RS is the model itself (pinned by the Markov enumeration); DT is an acceleration whose free
choices the paper does not fix, so this statistical agreement is the only thing that ties them to it.
Standard error: reading Q9 of P:101, sqrt((<x^2> - <x>^2) / (n - 1)).
Also a structural check: per sub-sweep the four colour passes cover every site exactly once.
"""
import numpy as np
import pytest


def sem(x):
    return np.sqrt((np.mean(x * x) - np.mean(x) ** 2) / (len(x) - 1))


def run(oracle_mod, L, N, R, S, K, times, seed, first_real=0):
    o = oracle_mod.Oracle(L, N, R, seed=seed, tile=S, subsweeps=K, first_real=first_real)
    out = {}
    t = 0
    for tt in times:
        o.advance(tt - t)
        t = tt
        W2, hm = o.width()
        out[tt] = (W2.copy(), hm.copy())
    o.close()
    return out


@pytest.mark.slow
@pytest.mark.parametrize("S,K", [(64, 1), (64, 4)])
def test_dt_matches_serial_rs(oracle_mod, S, K):
    """L = 128, N = 1, R = 1024 realizations each.  DT(64,4) must agree with serial RS within 3 combined
    standard errors at t = 10 and t = 100.  DT(64,1) (one origin per MCS, the paper's scheme verbatim,
    P:77) carries a known early-time bias of about -0.3 % in W2 that is unresolvable from t ~ 100 on
    (DESIGN.md "fidelity"): for it the 3-sigma test is applied at t = 100 and the t = 10
    deviation must lie in the band (-0.6 %, +0.1 %) around the measured bias of -0.24 % (
    combined SE here 0.09 %) -- far from the -3.5 % of 8x8 cells, which the next test checks is resolved.
    This is a COARSE regression bound at fixed seeds (R = 1024 resolves 0.3 %, not 0.03 %): it ties the free
    choices of the schedule to serial dynamics at that resolution and no finer; the high-precision bias
    table (R = 4096 per schedule) is DESIGN.md section 12."""
    L, N, R, times = 128, 1, 1024, (10, 100)
    # serial dynamics at L = 128: a tile side > L/2 selects RS
    rs = run(oracle_mod, L, N, R, 128, 1, times, seed=101)
    dt = run(oracle_mod, L, N, R, S, K, times, seed=202)
    for t in times:
        a, b = rs[t][0], dt[t][0]
        tol = 3.0 * np.sqrt(sem(a) ** 2 + sem(b) ** 2)
        assert tol < 0.02 * a.mean()                       # resolution: well below the 4 % bias of 8x8 cells
        if K == 1 and t < 100:
            d = (b.mean() - a.mean()) / a.mean()
            assert -0.006 < d < 0.001, (S, K, t, a.mean(), b.mean(), d)
        else:
            assert abs(a.mean() - b.mean()) <= tol, (S, K, t, a.mean(), b.mean(), tol)
        ha, hb = rs[t][1], dt[t][1]
        assert abs(ha.mean() - hb.mean()) <= 4.0 * np.sqrt(sem(ha) ** 2 + sem(hb) ** 2) + 2e-3 * ha.mean()
    # values agree with the survey's serial reference (0.63526(21), 1.7788(26))
    assert abs(rs[10][0].mean() - 0.63526) < 4 * sem(rs[10][0]) + 4 * 0.00021
    assert abs(rs[100][0].mean() - 1.7788) < 4 * sem(rs[100][0]) + 4 * 0.0026


@pytest.mark.slow
def test_the_test_has_teeth_small_cells_are_biased(oracle_mod):
    """8x8 sequential cells (the paper's finest domain) are measurably biased (-3.5 % in W2, SURVEY
    8c.4): the statistical test above must be able to see an effect of that size."""
    L, N, R, t = 128, 1, 512, 10
    rs = run(oracle_mod, L, N, R, 128, 1, (t,), seed=11)[t][0]
    d8 = run(oracle_mod, L, N, R, 8, 1, (t,), seed=12)[t][0]
    tol = 3.0 * np.sqrt(sem(rs) ** 2 + sem(d8) ** 2)
    assert rs.mean() - d8.mean() > tol
    assert 0.02 < (rs.mean() - d8.mean()) / rs.mean() < 0.05


@pytest.mark.parametrize("L,S,K", [(32, 8, 1), (64, 16, 2), (128, 64, 4)])
def test_each_subsweep_pass_covers_every_site_once(oracle_mod, L, S, K):
    """all four colours share the sub-sweep's origin, so the active tiles of one
    sub-sweep partition the lattice.  In the random-deposition limit (every attempt accepted) every
    S x S block of the origin-shifted tiling therefore gains exactly S^2/K deposits per sub-sweep, i.e.
    exactly S^2 per MCS only if K = 1; for any K the total is L^2 per MCS.  We recover the origin of
    a K = 1 sweep from the heights alone: exactly one shift makes all block sums equal S^2."""
    o = oracle_mod.Oracle(L, 10 ** 9, 2, seed=77, tile=S, subsweeps=K)
    o.advance(1)
    h = o.heights().astype(np.int64)
    o.close()
    assert (h.reshape(2, -1).sum(1) == L * L).all()
    if K != 1:
        return
    for r in range(2):
        shifts = []
        for oy in range(S):
            for ox in range(S):
                g = np.roll(h[r], (-oy, -ox), axis=(0, 1)).reshape(L // S, S, L // S, S).sum(axis=(1, 3))
                if (g == S * S).all():
                    shifts.append((ox, oy))
        assert len(shifts) == 1
