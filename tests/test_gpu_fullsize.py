"""GPU parity at BASELINE.json's full sizes, in the launch configuration `engine = auto` picks (the one bench.py
times): configs[4] (C5: every L in {64,128,256,512}, N in {1,2}, the config's own R), configs[2] at every N,
and the late ends of configs[1] and configs[3].  Run on the B200 with -m gpu.

Two kinds of check, both bit-exact (integers):
  prefix     realization r is a pure function of (seed, r, L, N, S, K): the oracle follows sampled realizations
             of the full run alone (first_real = r) from the flat start;
  induction  the GPU state at a late time t0 (a saturated / rough surface, |h| ~ 1e3..1e5) is handed to the oracle
             with set_state (t enters the Philox counter, so (heights, t) is the whole state); both advance and
             must agree.  With the exact prefixes this covers the run by induction on the sampled steps, and it is
             the test of the packed / mod-64 on-chip formats and of the anchor division far from the flat start.
No expected value comes from the CUDA path.
"""
import numpy as np
import pytest

from paper_1605_02620_b200.utils import workloads

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def rsos():
    import torch
    if not torch.cuda.is_available():
        pytest.skip("no CUDA device")
    from paper_1605_02620_b200 import build
    build.build()
    import paper_1605_02620_b200 as m
    return m


def _check_realization(g, gs, oracle_mod, cfg, r, t0, mcs, state=None):
    """Oracle follows realization r alone for `mcs` MCS (from the flat start, or from `state` = (heights, accepted)
    at time t0) and must equal the GPU's realization r (sums gs taken after the GPU advanced as well)."""
    o = oracle_mod.Oracle(cfg["L"], cfg["N"], 1, cfg["seed"], tile=cfg["tile"], subsweeps=cfg["subsweeps"], first_real=r)
    if state is not None:
        o.set_state(state[0], t0, state[1])
    o.advance(mcs)
    os1, os2, oacc = o.sums()
    assert (gs[0][r], gs[1][r], gs[2][r]) == (os1[0], os2[0], oacc[0]), "r=%d sums" % r
    hg, ho = g.heights(r, 1), o.heights()
    o.close()
    bad = np.argwhere(hg != ho)
    assert bad.size == 0, "r=%d heights differ at %d sites, first %s" % (r, len(bad), bad[:4].tolist())


def _c5(L, N):
    c = dict(workloads.CONFIGS["C5"])
    c.update(L=L, N=N, R=workloads.c5_realizations(L), mcs=workloads.c5_mcs(L))
    return c


@pytest.mark.parametrize("N", [1, 2])
@pytest.mark.parametrize("L", [64, 128, 256, 512])
def test_c5_full_size_prefix(rsos, oracle_mod, L, N):
    """configs[4]: the config's own R (4096 / 1024 / 256 / 64), DT(64,4) for L >= 128 (1024 tiles per colour pass),
    serial RS on chip for L = 64; three realizations followed alone by the oracle for 5 MCS from the flat start."""
    c = _c5(L, N)
    g = rsos.Rsos(L, N, c["R"], c["seed"], tile=c["tile"], subsweeps=c["subsweeps"])
    info = g.info()
    assert info["mode"] == ("RS" if L == 64 else "DT") and info["engine"] in ("onchip", "resident", "warp", "thread"), info
    g.advance(2)
    g.advance(3)
    gs = g.sums()
    assert (gs[0] == gs[2]).all()                            # sum h = accepted (flat start), every realization
    for r in (0, c["R"] // 2 + 1, c["R"] - 1):
        _check_realization(g, gs, oracle_mod, c, r, 0, 5)
    g.close()


@pytest.mark.parametrize("N", [1, 2])
@pytest.mark.parametrize("L", [64, 128, 256, 512])
def test_c5_full_size_saturated_induction(rsos, oracle_mod, L, N):
    """configs[4] at t0 = 0.75 * t_max (inside the config's measurement window, the stationary regime): two
    realizations go to the oracle, both sides advance 2 MCS.  Heights are ~ 0.3 * t0 (up to ~1e5 at L = 512)."""
    c = _c5(L, N)
    t0 = int(0.75 * c["mcs"])
    g = rsos.Rsos(L, N, c["R"], c["seed"], tile=c["tile"], subsweeps=c["subsweeps"])
    g.advance(t0)
    s1, s2, acc = g.sums()
    assert (s1 == acc).all()
    w2, hm = g.width()
    assert hm.min() > 0.2 * t0                              # grown far from the flat start
    assert w2.mean() > 0.08 * L ** 0.78, w2.mean()          # loose: a saturated width ~ 0.118 L^(2 alpha) at N = 1, more at N = 2
    picks = (1, c["R"] - 2)
    states = {}
    for r in picks:
        h0 = g.heights(r, 1)
        for ax in (0, 1):
            assert np.abs(h0[0] - np.roll(h0[0], 1, axis=ax)).max() <= N      # Eq. (6), periodic
        states[r] = (h0, acc[r:r + 1].copy())
    g.advance(2)
    gs = g.sums()
    for r in picks:
        _check_realization(g, gs, oracle_mod, c, r, t0, 2, states[r])
    g.close()


@pytest.mark.parametrize("N", [2, 3])
def test_c3_full_size_sampled_realizations_n23(rsos, oracle_mod, N):
    """configs[2] at N = 2 and 3 (N = 1 and 4 are in test_gpu_parity.py): 16384 tiles per pass, 4-bit sites."""
    c = dict(workloads.CONFIGS["C3"])
    c["N"] = N
    g = rsos.Rsos(c["L"], N, c["R"], c["seed"], tile=c["tile"], subsweeps=c["subsweeps"])
    assert g.info()["engine"] == "thread"
    g.advance(3)
    gs = g.sums()
    assert (gs[0] == gs[2]).all()
    for r in (0, 31, 63):
        _check_realization(g, gs, oracle_mod, c, r, 0, 3)
    g.close()


@pytest.mark.parametrize("N", [1, 2, 3, 4])
def test_c3_full_size_late_induction(rsos, oracle_mod, N):
    """configs[2] at its end: t0 = 4998, two realizations handed to the oracle, 2 MCS to t = 5000."""
    c = dict(workloads.CONFIGS["C3"])
    c["N"] = N
    t0 = c["mcs"] - 2
    g = rsos.Rsos(c["L"], N, c["R"], c["seed"], tile=c["tile"], subsweeps=c["subsweeps"])
    g.advance(t0)
    acc = g.sums()[2]
    states = {r: (g.heights(r, 1), acc[r:r + 1].copy()) for r in (5, 62)}
    g.advance(2)
    assert g.t == c["mcs"]
    gs = g.sums()
    for r, st in states.items():
        _check_realization(g, gs, oracle_mod, c, r, t0, 2, st)
    g.close()


def test_c2_full_size_induction_at_the_end(rsos, oracle_mod):
    """configs[1] at its end: t0 = 9998 of 10^4 MCS (all 128 realizations on the GPU), realizations 0, 64, 127."""
    c = dict(workloads.CONFIGS["C2"])
    t0 = c["mcs"] - 2
    g = rsos.Rsos(c["L"], c["N"], c["R"], c["seed"], tile=c["tile"], subsweeps=c["subsweeps"])
    g.advance(t0)
    acc = g.sums()[2]
    states = {r: (g.heights(r, 1), acc[r:r + 1].copy()) for r in (0, 64, 127)}
    for st in states.values():
        assert st[0].max() - st[0].min() > 12
    g.advance(2)
    assert g.t == c["mcs"]
    gs = g.sums()
    for r, st in states.items():
        _check_realization(g, gs, oracle_mod, c, r, t0, 2, st)
    g.close()


def test_c4_full_size_induction_at_the_end(rsos, oracle_mod):
    """configs[3] at its end: the whole 2^30-site surface at t0 = 1999 goes to the oracle; 1 MCS to t = 2000."""
    c = dict(workloads.CONFIGS["C4"])
    L, t0 = c["L"], c["mcs"] - 1
    g = rsos.Rsos(L, c["N"], 1, c["seed"], tile=c["tile"], subsweeps=c["subsweeps"])
    g.advance(t0)
    h0 = g.heights()
    acc = g.sums()[2]
    o = oracle_mod.Oracle(L, c["N"], 1, c["seed"], tile=c["tile"], subsweeps=c["subsweeps"])
    o.set_state(h0, t0, acc)
    del h0
    g.advance(1)
    o.advance(1)
    assert g.t == c["mcs"]
    assert all((a == b).all() for a, b in zip(g.sums(), o.sums()))
    hg = g.heights()
    g.close()
    ho = o.heights()
    o.close()
    assert np.array_equal(hg, ho)


@pytest.mark.parametrize("L,N,R,S,K,mcs", [(256, 3, 3, 64, 1, 6), (64, 1, 5, 64, 1, 40), (128, 2, 2, 64, 4, 9)])
def test_moments_equal_oracle(rsos, oracle_mod, L, N, R, S, K, mcs):
    """rsos_moments (exact 128-bit power sums about floor(mean)) and rsos_height_moments (Eq. 13) against the
    oracle's definitions on the same seeded run: integers exactly, doubles to 1e-12."""
    g = rsos.Rsos(L, N, R, 5, tile=S, subsweeps=K)
    o = oracle_mod.Oracle(L, N, R, 5, tile=S, subsweeps=K)
    g.advance(mcs)
    o.advance(mcs)
    base, M = g.moments()
    hbar, phi = g.height_moments()
    os1 = o.sums()[0]
    for r in range(R):
        assert int(base[r]) == int(os1[r]) // (L * L)
        assert M[r] == o.power_sums(r, int(base[r])), "r=%d power sums" % r
        ohb, ophi = o.height_moments(r)
        assert abs(hbar[r] - ohb) <= 1e-13 * max(1.0, abs(ohb))
        for k in range(3):
            assert abs(phi[r, k] - ophi[k]) <= 1e-12 * max(1.0, abs(ophi[k])), (r, k, phi[r, k], ophi[k])
    g.close()
    o.close()


def test_invalid_state_blocks_the_context(rsos):
    """after a rsos_set_state that violates Eq. (6) every engine-running or sum-reading call must fail
    until a valid state is set; a valid partial set_state elsewhere does not clear the mark."""
    for engine in (rsos.ENGINE_THREAD, rsos.ENGINE_WARP):
        g = rsos.Rsos(256, 1, 3, 1, engine=engine)
        g.advance(2)
        h = g.heights()
        acc = g.sums()[2]
        bad = h.copy()
        bad[1, 3, 4] += 5
        with pytest.raises(rsos.RsosError):
            g.set_state(bad[1:2], 2, acc[1:2], r0=1)
        for call in (lambda: g.advance(1), g.sums, g.width, g.moments, g.heights):
            with pytest.raises(rsos.RsosError) as e:
                call()
            assert e.value.code == -1
        with pytest.raises(rsos.RsosError):
            g.set_state(h[0:1], 2, acc[0:1], r0=0)          # valid, but realization 1 is still broken
        g.set_state(h[1:2], 2, acc[1:2], r0=1)              # repairs it: the whole lattice is valid again
        g.advance(1)
        assert (g.sums()[0] == g.sums()[2]).all()
        g.close()


@pytest.mark.parametrize("L,S,poisson", [(64, 8, False), (128, 8, False), (256, 16, False), (512, 8, False), (128, 8, True)])
def test_paper_cells_full_ensemble_sampled(rsos, oracle_mod, L, S, poisson):
    """The paper's steady-state setting (8 x 8 domains, L = 64 ... 512; 16 x 16) with BASELINE configs[4]'s
    ensemble sizes on the FINE engine (and its Poisson variant): three realizations of the full ensemble followed alone
    by the oracle for 4 MCS; then a saturated snapshot of two of them handed to the oracle."""
    R = workloads.c5_realizations(L)
    kw = dict(tile=S, poisson=True) if poisson else dict(tile=S, subsweeps=1)
    g = rsos.Rsos(L, 1, R, 1, **kw)
    assert g.info()["engine"] == "fine"
    g.advance(4)
    gs = g.sums()
    for r in (0, R // 2 + 1, R - 1):
        o = oracle_mod.Oracle(L, 1, 1, 1, first_real=r, **kw)
        o.advance(4)
        os1, os2, oacc = o.sums()
        assert (gs[0][r], gs[1][r], gs[2][r]) == (os1[0], os2[0], oacc[0])
        assert np.array_equal(g.heights(r, 1), o.heights())
        o.close()
    t0 = 4 + 600
    g.advance(600)
    for r in (1, R - 2):
        h, acc = g.heights(r, 1), g.sums()[2][r:r + 1]
        o = oracle_mod.Oracle(L, 1, 1, 1, first_real=r, **kw)
        o.set_state(h, t0, acc)
        o.advance(1)
        g2 = rsos.Rsos(L, 1, 1, 1, first_real=r, **kw)
        g2.set_state(h, t0, acc)
        g2.advance(1)
        assert np.array_equal(g2.heights(), o.heights()) and (g2.sums()[0] == o.sums()[0]).all()
        g2.close()
        o.close()
    g.close()


def test_multisurface_large_ensemble_sampled(rsos, oracle_mod):
    """opts.multisurface at L = 32 with 4096 realizations (32 groups of 128): members of different groups and warps
    followed alone by the oracle (a member is a pure function of its global index) for 5 MCS."""
    L, R = 32, 4096
    g = rsos.Rsos(L, 1, R, 2, multisurface=True)
    g.advance(5)
    gs = g.sums()
    for r in (0, 31, 32, 127, 128, 2049, 4095):
        o = oracle_mod.Oracle(L, 1, 1, 2, first_real=r, multisurface=True)
        o.advance(5)
        os1, os2, oacc = o.sums()
        assert (gs[0][r], gs[1][r], gs[2][r]) == (os1[0], os2[0], oacc[0]), r
        assert np.array_equal(g.heights(r, 1), o.heights()), r
        o.close()
    g.close()
