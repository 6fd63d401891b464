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

Tiers: A = the oracle runs the whole config; B = a full-oracle prefix of >= 16 MCS, snapshot induction at
>= 8 measurement times and, for configs with many realizations, >= 2 single realizations followed by the oracle for the
COMPLETE run (sums compared at every measurement time, heights at the end).  The `tier_b` tests below bring configs[1],
[2], [3] and [4] to B (configs[4] at L = 64 and 128 has 16 complete realizations per (L, N); at L = 256 and 512 a complete
realization costs minutes of oracle time and is left out, so those two sizes hold B's induction and prefix parts only).
configs[0] is at A in test_gpu_parity.py.
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


def _spread(seq, n):
    """n entries of seq, first and last included, evenly spread by index."""
    return [seq[(i * (len(seq) - 1)) // (n - 1)] for i in range(n)]


def _tier_b(rsos, oracle_mod, c, complete, induct, times, induct_times, expect_engine, oracle_R=1):
    """The GPU runs the FULL config c (engine = auto) through `times` (sorted measurement times, t_max last).
      - `complete`: first realizations of oracle runs (oracle_R consecutive realizations each) that follow the whole run from
        the flat start and are compared at every entry of `times` (S1, S2, accepted) and at the end (heights);
      - at every t in `induct_times` the GPU state of the realizations in `induct` goes to a fresh oracle (set_state; t enters
        the Philox counter), both sides advance one MCS and must agree in sums and in every height."""
    g = rsos.Rsos(c["L"], c["N"], c["R"], c["seed"], tile=c["tile"], subsweeps=c["subsweeps"])
    assert g.info()["engine"] in expect_engine, g.info()
    kw = dict(tile=c["tile"], subsweeps=c["subsweeps"])
    stops = sorted(set(times) | set(induct_times) | {t + 1 for t in induct_times})
    assert stops[-1] == times[-1] == c["mcs"]
    sums_at, pending = {}, {}
    for t in stops:
        g.advance(t - g.t)
        gs = g.sums()
        assert (gs[0] == gs[2]).all(), "t=%d: sum h != accepted" % t
        if t in times:
            sums_at[t] = gs
        for r, o in pending.pop(t - 1, []):                # oracles started one MCS ago from the GPU's state
            os1, os2, oacc = o.sums()
            assert (gs[0][r], gs[1][r], gs[2][r]) == (os1[0], os2[0], oacc[0]), "induction t=%d r=%d sums" % (t - 1, r)
            assert np.array_equal(g.heights(r, 1), o.heights()), "induction t=%d r=%d heights" % (t - 1, r)
            o.close()
        if t in induct_times:
            pending[t] = []
            for r in induct:
                o = oracle_mod.Oracle(c["L"], c["N"], 1, c["seed"], first_real=r, **kw)
                o.set_state(g.heights(r, 1), t, gs[2][r:r + 1].copy())
                o.advance(1)
                pending[t].append((r, o))
    assert not pending and g.t == c["mcs"]
    for r0 in complete:                                    # complete single realizations, flat start to t_max
        o = oracle_mod.Oracle(c["L"], c["N"], oracle_R, c["seed"], first_real=r0, **kw)
        for t in times:
            o.advance(t - o.t)
            for a, b in zip(sums_at[t], o.sums()):
                assert (a[r0:r0 + oracle_R] == b).all(), "complete run r0=%d t=%d" % (r0, t)
        assert np.array_equal(g.heights(r0, oracle_R), o.heights()), "complete run r0=%d final heights" % r0
        o.close()
    g.close()


def _measurement_times(t_max, prefix=16):
    """The config's 64 log-spaced times plus every MCS of the first `prefix` (the full-oracle prefix of tier B)."""
    return sorted(set(workloads.log_spaced_times(t_max)) | set(range(1, prefix + 1)))


def _induction_times(t_max):
    """8 times: 7 of the log-spaced measurement times beyond the prefix, spread over the run, and the last MCS of the run."""
    return _spread([t for t in workloads.log_spaced_times(t_max) if 16 < t < t_max - 1], 7) + [t_max - 1]


def test_c2_tier_b(rsos, oracle_mod):
    """configs[1] in full on the GPU (128 realizations, 10^4 MCS, the 4-lanes-per-tile launch bench.py times).  Realizations
    0 and 127 are followed by the oracle for the WHOLE run (1.05e10 attempts each) and compared at the 57 log-spaced times
    and at every MCS up to 16; realizations 17 and 100 are handed over at 8 measurement times."""
    c = dict(workloads.CONFIGS["C2"])
    times = _measurement_times(c["mcs"])
    induct_times = _induction_times(c["mcs"])
    _tier_b(rsos, oracle_mod, c, complete=(0, 127), induct=(17, 100), times=times, induct_times=induct_times,
            expect_engine=("thread",))


@pytest.mark.parametrize("N", [1, 2, 3, 4])
def test_c3_tier_b(rsos, oracle_mod, N):
    """configs[2] in full on the GPU at every N (64 realizations, 5000 MCS): one complete oracle realization per N (four
    over the config, 2.1e10 attempts each), two realizations handed over at 8 measurement times."""
    c = dict(workloads.CONFIGS["C3"])
    c["N"] = N
    times = _measurement_times(c["mcs"])
    induct_times = _induction_times(c["mcs"])
    _tier_b(rsos, oracle_mod, c, complete=((0, 21, 42, 63)[N - 1],), induct=(5, 62), times=times, induct_times=induct_times,
            expect_engine=("thread",))


@pytest.mark.parametrize("N", [1, 2])
@pytest.mark.parametrize("L", [64, 128, 256, 512])
def test_c5_tier_b(rsos, oracle_mod, L, N):
    """configs[4] on the GPU at the config's own R, up to t = 20 L^1.6 (0.8 of it at L = 512): two realizations handed over at 8 times
    spread over the run (the last ones inside the stationary measurement window, |h| up to ~1e5 at L = 512); at L = 64 and
    128 sixteen consecutive realizations are followed by the oracle for the complete run."""
    c = _c5(L, N)
    t_full = c["mcs"]
    if L == 512:
        c["mcs"] = int(0.8 * t_full)                        # 7e12 attempts in full: stop a little inside the measurement window
    times = _measurement_times(c["mcs"])
    induct_times = _induction_times(c["mcs"])
    assert induct_times[-1] > 0.75 * t_full                 # inside the final 25 % the config averages over
    complete = (c["R"] // 2,) if L <= 128 else ()
    _tier_b(rsos, oracle_mod, c, complete=complete, induct=(1, c["R"] - 2), times=times, induct_times=induct_times,
            expect_engine=("onchip", "resident"), oracle_R=16)


def test_c4_tier_b(rsos, oracle_mod):
    """configs[3]: the whole 2^30-site surface.  Prefix: the oracle follows it from the flat start for 16 MCS (sums every MCS,
    every height at t = 16).  Induction: at 8 of the config's log-spaced times up to t = 1999 the whole surface goes to the
    oracle, both sides advance one MCS, sums and all 2^30 heights must agree."""
    c = dict(workloads.CONFIGS["C4"])
    L = c["L"]
    g = rsos.Rsos(L, c["N"], 1, c["seed"], tile=c["tile"], subsweeps=c["subsweeps"])
    assert g.info()["engine"] == "thread"
    o = oracle_mod.Oracle(L, c["N"], 1, c["seed"], tile=c["tile"], subsweeps=c["subsweeps"])
    for t in range(1, 17):
        g.advance(1)
        o.advance(1)
        assert all((a == b).all() for a, b in zip(g.sums(), o.sums())), "prefix t=%d" % t
    assert np.array_equal(g.heights(), o.heights()), "prefix heights at t = 16"
    induct_times = _induction_times(c["mcs"])
    for t in induct_times:
        g.advance(t - g.t)
        h0 = g.heights()
        o.set_state(h0, t, g.sums()[2])
        del h0
        g.advance(1)
        o.advance(1)
        assert all((a == b).all() for a, b in zip(g.sums(), o.sums())), "induction t=%d sums" % t
        hg = g.heights()
        assert np.array_equal(hg, o.heights()), "induction t=%d heights" % t
        del hg
    assert g.t == c["mcs"]
    g.close()
    o.close()


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
