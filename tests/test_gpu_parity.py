"""GPU parity (run on the B200 with -m gpu): the CUDA path behind the C ABI against the CPU oracle.

Integer work, so the bar is bit-exact: heights element by element, and (S1, S2, accepted) exactly
(BASELINE.json north_star).  Both sides execute the seeded schedule of DESIGN.md section 2 on the
same (L, N, R, seed, S, K); no expected value comes from the CUDA path.
"""
import numpy as np
import pytest

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


def compare(g, o, what=""):
    gs1, gs2, gacc = g.sums()
    os1, os2, oacc = o.sums()
    assert (gs1 == os1).all(), what + " S1"
    assert (gs2 == os2).all(), what + " S2"
    assert (gacc == oacc).all(), what + " accepted"
    hg, ho = g.heights(), o.heights()
    bad = np.argwhere(hg != ho)
    assert bad.size == 0, "%s heights differ at %d sites, first %s" % (what, len(bad), bad[:5].tolist())
    gw, gh = g.width()
    ow, oh = o.width()
    assert (gw == ow).all() and (gh == oh).all(), what + " W2/hmean doubles"


def test_philox_device_equals_oracle(rsos, oracle_mod):
    rng = np.random.default_rng(3)
    n = 20000
    ctr = rng.integers(0, 2 ** 32, size=(n, 4), dtype=np.uint64).astype(np.uint32)
    key = rng.integers(0, 2 ** 32, size=(n, 2), dtype=np.uint64).astype(np.uint32)
    ctr[0] = 0; key[0] = 0
    ctr[1] = 0xFFFFFFFF; key[1] = 0xFFFFFFFF
    out = rsos.philox(ctr, key)
    assert out[0].tolist() == [0x6627e8d5, 0xe169c58d, 0xbc57ac4c, 0x9b00dbd8]      # tests/golden/philox_kat.txt
    assert out[1].tolist() == [0x408f276d, 0x41c83b0e, 0xa20bc7c6, 0x6d5451fd]
    for i in range(0, n, 7):
        assert (out[i] == oracle_mod.philox(ctr[i], key[i])).all()


@pytest.mark.parametrize("engine", ["auto", "onchip", "simple"])
def test_c1_full_config_every_mcs(rsos, oracle_mod, engine):
    """BASELINE.json configs[0]: L=32, N=1, R=128, 100 MCS, seed 1, sums at every MCS (tier A).  engine = auto is the
    LEVEL engine (few realizations), the launch configuration bench.py times."""
    eng = {"auto": rsos.ENGINE_AUTO, "onchip": rsos.ENGINE_ONCHIP, "simple": rsos.ENGINE_SIMPLE}[engine]
    g = rsos.Rsos(32, 1, 128, 1, engine=eng)
    o = oracle_mod.Oracle(32, 1, 128, 1)
    assert g.info()["mode"] == "RS" and o.mode == "RS"
    for t in range(100):
        g.advance(1)
        o.advance(1)
        gs, os_ = g.sums(), o.sums()
        assert all((a == b).all() for a, b in zip(gs, os_)), "t=%d" % (t + 1)
    compare(g, o, "C1 " + engine)
    g.close()


@pytest.mark.parametrize("L,N,R,S,K,mcs,seed", [
    (128, 1, 3, 64, 1, 6, 1),        # smallest DT lattice at the default tile: T = 2, one tile per colour
    (256, 1, 2, 64, 1, 5, 2),        # several tiles, wrap-around windows
    (256, 2, 2, 64, 4, 4, 3),        # K = 4 sub-sweeps
    (256, 4, 1, 64, 1, 4, 4),        # larger slopes (config C3)
    (512, 3, 1, 64, 2, 3, 5),
    (128, 1, 2, 32, 4, 5, 6),        # S = 32
    (64, 2, 3, 16, 1, 5, 7),         # S = 16
    (64, 1, 2, 8, 2, 5, 8),          # S = 8, A = 32 attempts per tile
    (256, 1, 1, 128, 1, 3, 9),       # S = 128
    (128, 31, 1, 64, 1, 3, 10),      # largest N of the 6-bit on-chip format
    (128, 1, 1, 64, 128, 2, 11),     # A = 32: a single window per tile
])
def test_dt_warp_engine_equals_oracle(rsos, oracle_mod, L, N, R, S, K, mcs, seed):
    g = rsos.Rsos(L, N, R, seed, tile=S, subsweeps=K, engine=rsos.ENGINE_WARP)
    o = oracle_mod.Oracle(L, N, R, seed, tile=S, subsweeps=K)
    assert g.info()["mode"] == "DT" and o.mode == "DT"
    for step in range(mcs):
        g.advance(1)
        o.advance(1)
        compare(g, o, "DT warp L=%d N=%d S=%d K=%d t=%d" % (L, N, S, K, step + 1))
    g.close()


@pytest.mark.parametrize("L,N,R,S,K,mcs,seed", [
    (128, 1, 3, 64, 1, 6, 1),        # one tile per colour per realization: 3 live lanes, 29 idle ones
    (256, 1, 5, 64, 1, 5, 2),        # lanes of one warp span realizations with different origins
    (512, 1, 3, 64, 1, 4, 12),       # 48 tiles per pass: two warps, ragged tail
    (256, 2, 2, 64, 4, 4, 3),        # 4-bit sites (N = 2), K = 4 sub-sweeps
    (256, 4, 1, 64, 1, 4, 4),        # config C3 slopes
    (512, 7, 1, 64, 2, 3, 5),        # largest N of the 4-bit format
    (128, 1, 2, 32, 4, 5, 6),        # S = 32
    (64, 2, 3, 16, 1, 5, 7),         # S = 16
    (64, 1, 2, 8, 2, 5, 8),          # S = 8, A = 32 attempts per tile
    (128, 1, 1, 64, 128, 2, 11),     # A = 32
])
@pytest.mark.parametrize("lanes", [1, 2, 4, 8])
def test_dt_thread_engine_equals_oracle(rsos, oracle_mod, L, N, R, S, K, mcs, seed, lanes):
    """The lane-per-tile engine (2- or 4-bit sites, bank-interleaved shared memory), 1, 2, 4 or 8 lanes per tile."""
    if 8 * lanes > S * S // K:
        pytest.skip("a batch of 8 * lanes attempts does not fit the tile")
    g = rsos.Rsos(L, N, R, seed, tile=S, subsweeps=K, engine=rsos.ENGINE_THREAD, lanes=lanes)
    o = oracle_mod.Oracle(L, N, R, seed, tile=S, subsweeps=K)
    assert g.info()["mode"] == "DT" and g.info()["engine"] == "thread"
    for step in range(mcs):
        g.advance(1)
        o.advance(1)
        compare(g, o, "DT thread L=%d N=%d S=%d K=%d t=%d" % (L, N, S, K, step + 1))
    g.close()


@pytest.mark.parametrize("L,N,R,S,K,mcs,seed", [
    (128, 1, 3, 64, 1, 6, 1),        # one tile per colour pass and realization: one warp per block, no cluster
    (128, 1, 9, 64, 4, 5, 21),       # C5's shape at L = 128 (K = 4): 1024 attempts per tile and pass
    (256, 1, 5, 64, 4, 4, 2),        # 4 tiles per pass: 4 warps in one block .. 4 blocks of one warp
    (512, 1, 2, 64, 4, 3, 12),       # 16 tiles per pass, 256 KiB of uint8 sites: needs a cluster of >= 2 blocks
    (256, 2, 2, 64, 4, 4, 3),        # 4-bit sites (N = 2): uint16 on chip
    (512, 2, 1, 64, 4, 2, 14),       # 512 KiB of uint16 sites: a cluster of >= 4 blocks
    (256, 4, 1, 64, 1, 4, 4),
    (256, 7, 1, 64, 2, 3, 5),        # largest N of the 4-bit format
    (128, 1, 2, 32, 4, 5, 6),        # S = 32, A = 256 attempts
    (256, 3, 2, 32, 1, 3, 16),       # S = 32, 16 tiles per pass
    (64, 2, 3, 16, 1, 5, 7),         # S = 16
    (64, 1, 5, 16, 2, 5, 8),         # S = 16, 2-bit sites, A = 128
    (128, 1, 2, 64, 128, 3, 11),     # A = 32: a single window per tile and pass
    (1024, 1, 1, 64, 1, 2, 17),      # 64 tiles per pass: 8 or 16 blocks of 8 or 4 warps, rows fetched across the cluster
])
@pytest.mark.parametrize("cluster", [0, 1, 2, 4, 8, 16])
def test_dt_resident_engine_equals_oracle(rsos, oracle_mod, L, N, R, S, K, mcs, seed, cluster):
    """The RESIDENT engine: lattice in the shared memory of a cluster of 1 .. 16 thread blocks across all passes of a
    call, one warp per tile with 32 attempts in flight and exact conflict votes (rsos_resident.cu)."""
    try:
        want = rsos.plan(L, N, R, tile=S, subsweeps=K, engine=rsos.ENGINE_RESIDENT, cluster=cluster)
    except rsos.RsosError as e:
        assert e.code == -5
        pytest.skip("cluster size %d does not fit this shape" % cluster)
    g = rsos.Rsos(L, N, R, seed, tile=S, subsweeps=K, engine=rsos.ENGINE_RESIDENT, cluster=cluster)
    o = oracle_mod.Oracle(L, N, R, seed, tile=S, subsweeps=K)
    info = g.info()
    assert info["mode"] == "DT" and info["engine"] == "resident" and info["cluster"] == want["cluster"], info
    assert cluster == 0 or info["cluster"] == cluster
    assert not info["int32_allocated"]                      # the int32 lattice exists only on demand
    for step in (1, 1, mcs - 2):                            # single MCS and several MCS inside one launch
        g.advance(step)
        o.advance(step)
        compare(g, o, "DT resident L=%d N=%d S=%d K=%d cluster=%d t=%d" % (L, N, S, K, cluster, g.t))
    g.close()


def test_dt_resident_engine_snapshot_restart(rsos, oracle_mod):
    """RESIDENT engine: packed working state, heights read back mid-run, a partial rsos_set_state, many MCS per launch."""
    L, N, R, seed = 128, 1, 6, 41
    g = rsos.Rsos(L, N, R, seed, subsweeps=4)
    assert g.info()["engine"] == "resident"
    o = oracle_mod.Oracle(L, N, R, seed, subsweeps=4)
    g.advance(40)
    o.advance(40)
    compare(g, o, "before snapshot")
    h, acc = o.heights(), o.sums()[2]
    g.set_state(h[2:4], 40, acc[2:4], r0=2)
    g.advance(25)
    o.advance(25)
    compare(g, o, "after partial set_state")
    g.close()


@pytest.mark.parametrize("L,N,R,mcs", [(2048, 1, 2, 2),     # 512 tiles per pass; rows rebuilt by one warp each
                                       (4096, 1, 1, 1),     # 256 packed words per row: rows rebuilt by a whole block
                                       (2048, 3, 1, 1)])    # 4-bit sites, 256 words per row
@pytest.mark.parametrize("lanes", [0, 2])
def test_dt_thread_engine_large_lattices(rsos, oracle_mod, L, N, R, mcs, lanes):
    """Many tiles per pass and both row-team shapes of the packed -> int32 rebuild (rsos_pack.cu)."""
    g = rsos.Rsos(L, N, R, 13, engine=rsos.ENGINE_THREAD, lanes=lanes)
    o = oracle_mod.Oracle(L, N, R, 13)
    g.advance(mcs)
    o.advance(mcs)
    compare(g, o, "DT thread L=%d N=%d" % (L, N))
    g.close()


def test_dt_thread_engine_snapshot_restart(rsos, oracle_mod):
    """Packed working lattice: heights read back mid-run, a snapshot written into SOME realizations
    (rsos_set_state) and the run continued; every realization must still follow the oracle."""
    L, N, R, seed = 256, 1, 4, 31
    g = rsos.Rsos(L, N, R, seed, engine=rsos.ENGINE_THREAD)
    o = oracle_mod.Oracle(L, N, R, seed)
    g.advance(3)
    o.advance(3)
    compare(g, o, "before snapshot")
    h = o.heights()
    acc = o.sums()[2]
    g2 = rsos.Rsos(L, N, R, seed, engine=rsos.ENGINE_THREAD)
    g2.advance(1)                                           # some other state, to be overwritten
    g2.set_state(h, 3, acc)
    g.set_state(h[1:3], 3, acc[1:3], r0=1)                  # rewrite realizations 1, 2 with their own state
    for x in (g, g2):
        x.advance(2)
    o.advance(2)
    compare(g, o, "after partial set_state")
    compare(g2, o, "restart from snapshot")
    g.close()
    g2.close()


@pytest.mark.parametrize("L,N,R,S,K,mcs", [(128, 1, 2, 64, 1, 3), (128, 2, 2, 16, 4, 3), (1024, 1, 1, 512, 1, 1),
                                           (128, 40, 1, 64, 1, 2)])
def test_dt_simple_engine_equals_oracle(rsos, oracle_mod, L, N, R, S, K, mcs):
    g = rsos.Rsos(L, N, R, 21, tile=S, subsweeps=K, engine=rsos.ENGINE_SIMPLE if N <= 31 else rsos.ENGINE_AUTO)
    assert g.info()["engine"] == "simple"
    o = oracle_mod.Oracle(L, N, R, 21, tile=S, subsweeps=K)
    g.advance(mcs)
    o.advance(mcs)
    compare(g, o, "DT simple")
    g.close()


@pytest.mark.parametrize("L,N,R,mcs", [(4, 1, 5, 30), (8, 2, 33, 20), (16, 1, 7, 20), (64, 1, 9, 12), (64, 3, 4, 12),
                                       (128, 1, 3, 5), (32, 31, 2, 40)])
def test_rs_onchip_engine_equals_oracle(rsos, oracle_mod, L, N, R, mcs):
    """RS mode (2S > L): serial random-sequential dynamics with the whole lattice on chip."""
    g = rsos.Rsos(L, N, R, 5, tile=128, engine=rsos.ENGINE_ONCHIP)
    o = oracle_mod.Oracle(L, N, R, 5, tile=128)
    assert g.info()["mode"] == "RS" and o.mode == "RS"
    g.advance(3)                      # several sweeps inside one launch ...
    g.advance(mcs - 3)                # ... and a second call continuing from the stored heights
    o.advance(mcs)
    compare(g, o, "RS onchip L=%d N=%d" % (L, N))
    g.close()


def test_rs_simple_large_lattice_32bit_slots(rsos, oracle_mod):
    """RS with L = 512: 2 lg L > 16 selects the 32-bit slot layout (4 slots per Philox call)."""
    g = rsos.Rsos(512, 1, 2, 9, tile=512)
    assert g.info() ["engine"] == "simple" and g.info()["mode"] == "RS"
    o = oracle_mod.Oracle(512, 1, 2, 9, tile=512)
    g.advance(1)
    o.advance(1)
    compare(g, o, "RS simple L=512")
    g.close()


def test_first_real_splits_a_run(rsos, oracle_mod):
    """Realization r is a pure function of (seed, r, ...): contexts with first_real offsets tile a run."""
    o = oracle_mod.Oracle(128, 1, 4, 77)
    o.advance(3)
    ho = o.heights()
    for r0 in (0, 1, 3):
        g = rsos.Rsos(128, 1, 1, 77, first_real=r0)
        g.advance(3)
        assert (g.heights()[0] == ho[r0]).all()
        g.close()


def test_snapshot_restart_and_state_roundtrip(rsos, oracle_mod):
    """rsos_set_state: (heights, t) is the whole state because t sits in the Philox counter."""
    a = rsos.Rsos(256, 2, 2, 13)
    a.advance(5)
    snap = a.heights()
    _, _, acc = a.sums()
    a.advance(2)
    b = rsos.Rsos(256, 2, 2, 13)
    b.set_state(snap, 5, acc)
    assert b.t == 5
    b.advance(2)
    assert (a.heights() == b.heights()).all()
    assert all((x == y).all() for x, y in zip(a.sums(), b.sums()))
    o = oracle_mod.Oracle(256, 2, 2, 13)
    o.set_state(snap, 5, acc)
    o.advance(2)
    compare(b, o, "snapshot")
    a.close(); b.close()


def test_borrowed_torch_buffer_and_stream(rsos, oracle_mod):
    import torch
    L, R = 128, 2
    buf = torch.full((R, L, L), 7, dtype=torch.int32, device="cuda")     # content ignored: flat start
    st = torch.cuda.Stream()
    g = rsos.Rsos(L, 1, R, 3, d_heights=buf.data_ptr(), stream=st.cuda_stream)
    assert g.device_heights() == buf.data_ptr()
    g.advance(4)
    o = oracle_mod.Oracle(L, 1, R, 3)
    o.advance(4)
    compare(g, o, "borrowed buffer")
    st.synchronize()
    assert (buf.cpu().numpy() == o.heights()).all()
    g.close()


def test_invariants_on_device_result(rsos, oracle_mod):
    """Eq. (6) holds on every bond, heights never decrease, sum h == accepted (pins P1-P3 on the GPU state)."""
    g = rsos.Rsos(256, 2, 3, 99)
    prev = g.heights()
    for _ in range(4):
        g.advance(2)
        h = g.heights()
        assert (h >= prev).all()
        for r in range(3):
            assert oracle_mod.violations(h[r], 2) == 0
        S1, S2, acc = g.sums()
        assert (S1 == acc).all()
        assert (S1 == h.reshape(3, -1).astype(np.int64).sum(1)).all()
        assert (S2 == (h.reshape(3, -1).astype(np.int64) ** 2).sum(1).astype(np.uint64)).all()
        prev = h
    g.close()


@pytest.mark.parametrize("engine", ["auto", "thread"])
def test_moments_exact(rsos, engine):
    """rsos_moments right after rsos_advance: with the THREAD engine it has to rebuild the int32 heights first."""
    g = rsos.Rsos(256, 3, 2, 5, engine=rsos.ENGINE_THREAD if engine == "thread" else rsos.ENGINE_AUTO)
    g.advance(6)
    base, M = g.moments()
    h = g.heights()
    for r in range(2):
        d = [int(v) - int(base[r]) for v in h[r].ravel()]
        assert int(base[r]) == sum(int(v) for v in h[r].ravel()) // (256 * 256)
        for k in range(4):
            assert M[r][k] == sum(x ** (k + 1) for x in d)
    g.close()


def test_error_paths(rsos):
    for args, kw in [((3, 1, 1, 1), {}), ((65537, 1, 1, 1), {}), ((64, 0, 1, 1), {}), ((64, 1, 0, 1), {}), ((64, 200, 1, 1), {}),
                     ((128, 1, 1, 1), dict(tile=24)), ((128, 1, 1, 1), dict(tile=8, subsweeps=4)),
                     ((128, 1, 1, 1), dict(subsweeps=3))]:
        with pytest.raises(rsos.RsosError) as e:
            rsos.Rsos(*args, **kw)
        assert e.value.code == -1
    with pytest.raises(rsos.RsosError) as e:
        rsos.Rsos(64, 1, 1, 1, engine=rsos.ENGINE_WARP)          # RS mode cannot use the DT warp engine
    assert e.value.code == -5
    g = rsos.Rsos(128, 1, 1, 1, subsweeps=4)
    with pytest.raises(rsos.RsosError) as e:
        g.advance(2 ** 30)                                           # (t + mcs) * K reaches 2^32
    assert e.value.code == -2 and g.t == 0
    with pytest.raises(rsos.RsosError):
        g.heights(r0=1, nr=1)
    g.advance(0)
    assert g.t == 0
    g.close()


# ---------------------------------------------------------------------------------------------
# Full-size configurations in the launch configuration bench.py times (engine auto, default lanes),
# compared on sampled outputs the oracle can compute one by one: realization r is a pure function
# of (seed, r, ...), so the oracle follows single realizations of the full run (first_real = r).
# ---------------------------------------------------------------------------------------------
def _sampled_realizations(rsos, oracle_mod, cfg, N, mcs, sample, want_engine, want_lanes):
    from paper_1605_02620_b200.utils import workloads
    c = dict(workloads.CONFIGS[cfg])
    g = rsos.Rsos(c["L"], N, c["R"], c["seed"], tile=c["tile"], subsweeps=c["subsweeps"])
    info = g.info()
    assert info["engine"] == want_engine and info["lanes"] == want_lanes, info
    g.advance(mcs)
    gs1, gs2, gacc = g.sums()                               # from the packed lattice, all realizations
    for r in sample:
        o = oracle_mod.Oracle(c["L"], N, 1, c["seed"], tile=c["tile"], subsweeps=c["subsweeps"], first_real=r)
        o.advance(mcs)
        os1, os2, oacc = o.sums()
        assert (gs1[r], gs2[r], gacc[r]) == (os1[0], os2[0], oacc[0]), "%s r=%d sums" % (cfg, r)
        assert np.array_equal(g.heights(r, 1), o.heights()), "%s r=%d heights" % (cfg, r)
        o.close()
    # properties that hold for every realization at any size
    assert (gs1 == gacc).all()                              # sum h = accepted deposits (flat start)
    h = g.heights(0, 1)[0]
    for ax in (0, 1):
        assert np.abs(h - np.roll(h, 1, axis=ax)).max() <= N    # Eq. (6) on every bond, periodic
    g.close()


def test_c2_full_size_sampled_realizations(rsos, oracle_mod):
    """BASELINE.json configs[1] (L=1024, N=1, R=128): 8192 tiles per pass, THREAD engine, 4 lanes per tile."""
    _sampled_realizations(rsos, oracle_mod, "C2", 1, 6, [0, 77, 127], "thread", 4)


@pytest.mark.parametrize("N", [1, 4])
def test_c3_full_size_sampled_realizations(rsos, oracle_mod, N):
    """configs[2] (L=2048, R=64, N in 1..4): 16384 tiles per pass, 2 lanes per tile; N=4 uses 4-bit sites."""
    _sampled_realizations(rsos, oracle_mod, "C3", N, 3, [0, 63], "thread", 2 if N == 1 else 4)


def test_c4_full_size_whole_surface(rsos, oracle_mod):
    """configs[3] (L=32768, N=1, R=1, 4 GiB of int32 heights): the whole surface after 2 MCS (2.1e9 attempts),
    element by element, plus the exact sums taken from the packed lattice."""
    L = 32768
    g = rsos.Rsos(L, 1, 1, 1)
    assert g.info()["engine"] == "thread" and g.info()["lanes"] == 2
    o = oracle_mod.Oracle(L, 1, 1, 1)
    g.advance(2)
    o.advance(2)
    assert all((a == b).all() for a, b in zip(g.sums(), o.sums()))
    hg = g.heights()
    g.close()
    ho = o.heights()
    o.close()
    assert np.array_equal(hg, ho)


# ---------------------------------------------------------------------------------------------
# Snapshot induction at late times (rough surfaces), full size: the GPU state at time t is handed to
# the oracle (t enters the Philox counter, so (heights, t) is the whole state), both advance, and
# the results must be equal.  Together with the exact prefixes above this covers the whole run by
# induction on the sampled steps.
# ---------------------------------------------------------------------------------------------
@pytest.mark.parametrize("t0", [300, 1500])
def test_c2_full_size_snapshot_induction(rsos, oracle_mod, t0):
    """C2 in full (128 realizations, bench launch configuration): realizations 3 and 126 at time t0 go to the
    oracle, the full GPU run and the oracle both advance 2 MCS, and those realizations must be equal."""
    from paper_1605_02620_b200.utils import workloads
    c = dict(workloads.CONFIGS["C2"])
    g = rsos.Rsos(c["L"], c["N"], c["R"], c["seed"], tile=c["tile"], subsweeps=c["subsweeps"])
    assert g.info()["engine"] == "thread"
    g.advance(t0)
    acc = g.sums()[2]
    oracles = {}
    for r in (3, 126):
        h0 = g.heights(r, 1)
        for ax in (0, 1):
            assert np.abs(h0[0] - np.roll(h0[0], 1, axis=ax)).max() <= c["N"]
        assert h0.max() - h0.min() > 8                      # a rough surface, not the flat start
        o = oracle_mod.Oracle(c["L"], c["N"], 1, c["seed"], tile=c["tile"], subsweeps=c["subsweeps"], first_real=r)
        o.set_state(h0, t0, acc[r:r + 1])
        o.advance(2)
        oracles[r] = o
    g.advance(2)
    gs1, gs2, gacc = g.sums()
    for r, o in oracles.items():
        os1, os2, oacc = o.sums()
        assert (gs1[r], gs2[r], gacc[r]) == (os1[0], os2[0], oacc[0]), "r=%d sums" % r
        assert np.array_equal(g.heights(r, 1), o.heights()), "r=%d heights" % r
        o.close()
    g.close()


def test_c4_full_size_snapshot_induction(rsos, oracle_mod):
    """C4: the whole 2^30-site surface at t = 40 goes to the oracle; both advance 1 MCS; all heights equal."""
    L = 32768
    g = rsos.Rsos(L, 1, 1, 1)
    g.advance(40)
    h0 = g.heights()
    acc = g.sums()[2]
    o = oracle_mod.Oracle(L, 1, 1, 1)
    o.set_state(h0, 40, acc)
    del h0
    g.advance(1)
    o.advance(1)
    assert all((a == b).all() for a, b in zip(g.sums(), o.sums()))
    hg = g.heights()
    g.close()
    ho = o.heights()
    o.close()
    assert np.array_equal(hg, ho)


def test_dd_consistency_table_on_gpu(rsos):
    """SURVEY 8(f) NEXT-1 / DESIGN.md section 12: the tile side sets the bias of the decomposed schedule against
    serial RS ("domain size ... noise amplitude").  Deterministic (fixed seeds); values recorded in DESIGN.md."""
    from paper_1605_02620_b200 import dd_consistency
    rows = dd_consistency.table(L=128, N=1, R=4096, seed=1, times=(1, 10, 100))
    dev = {name: d for name, _, _, d, _ in rows if d is not None}
    eng = {name: e for name, e, _, _, _ in rows}
    assert eng["DT(8,1)"] == eng["DT(16,1)"] == eng["DTP(8)"] == "fine"
    bias_t1 = [abs(dev["DT(%d,1)" % S][0][0]) for S in (8, 16, 32, 64)]
    assert bias_t1 == sorted(bias_t1, reverse=True) and bias_t1[0] > 0.03 > 0.006 > bias_t1[3]
    for i in range(3):                                      # the fidelity setting agrees with serial dynamics
        dw, sdw, dh, sdh = dev["DT(64,4)"][i]
        assert abs(dw) < 4 * sdw and abs(dh) < 5e-4
    dw, sdw, _, _ = dev["DT(64,1)"][2]                      # the default: unresolvable from t ~ 100 on
    assert abs(dw) < 3 * sdw
    for name in ("DTP(8)", "DTP(16)"):                      # the Poisson variant of the paper's small cells agrees with
        for i in range(3):                                  # serial dynamics (S 8(c).4), where fixed counts are 1.6-3.6 % low
            dw, sdw, dh, sdh = dev[name][i]
            assert abs(dw) < 4.5 * sdw and abs(dh) < 4.5 * sdh, (name, i, dw, sdw, dh, sdh)


def test_growth_exponent_sanity_c2(rsos):
    """Loose physics pin P10 (not parity): on C2 the slope of ln<W^2> vs ln t over t in [100, 3200] is 2 beta with
    beta = 0.241(1) in the paper.  Measured on the B200: 0.4754."""
    from paper_1605_02620_b200.utils import workloads
    c = dict(workloads.CONFIGS["C2"])
    g = rsos.Rsos(c["L"], c["N"], c["R"], c["seed"], tile=c["tile"], subsweeps=c["subsweeps"])
    ts, t, w = [100, 200, 400, 800, 1600, 3200], 0, []
    for tt in ts:
        g.advance(tt - t)
        t = tt
        w.append(g.width()[0].mean())
    g.close()
    slope = np.polyfit(np.log(ts), np.log(w), 1)[0]
    assert 0.45 < slope < 0.50, slope


def test_set_state_rejects_surfaces_that_violate_eq6(rsos):
    """rsos_set_state checks Eq. (6) on the device (all engines rely on it): one bad bond -> RSOS_EINVAL."""
    for engine in (rsos.ENGINE_THREAD, rsos.ENGINE_WARP):
        g = rsos.Rsos(256, 2, 3, 1, engine=engine)
        g.advance(2)
        h = g.heights()
        acc = g.sums()[2]
        g.set_state(h, 2, acc)                              # its own state: fine
        bad = h.copy()
        bad[1, 17, 255] += 3                                # wraps to column 0: periodic bonds are checked too
        with pytest.raises(rsos.RsosError) as e:
            g.set_state(bad, 2, acc)
        assert e.value.code == -1 and "Eq. (6)" in str(e.value)
        g.set_state(h, 2, acc)                              # recover
        g.advance(1)
        assert (g.sums()[0] == g.sums()[2]).all()
        g.close()


def test_random_shapes_all_dt_engines(rsos, oracle_mod):
    """Seeded random sweep over (L, N, R, S, K, engine, lanes): every DT engine against the oracle."""
    rng = np.random.default_rng(20261104)
    done = 0
    while done < 24:
        S = int(rng.choice([8, 16, 32, 64]))
        L = int(S * rng.choice([2, 4, 8]))
        if L > 512:
            continue
        K = int(rng.choice([k for k in (1, 2, 4, 8, 16) if S * S // k >= 32]))
        N = int(rng.choice([1, 1, 2, 3, 5, 7]))
        R = int(rng.integers(1, 6))
        seed = int(rng.integers(1, 2 ** 40))
        first = int(rng.integers(0, 1000))
        lanes = int(rng.choice([l for l in (1, 2, 4, 8) if 8 * l <= S * S // K]))
        engines = [(rsos.ENGINE_THREAD, lanes), (rsos.ENGINE_WARP, 0)]
        if S >= 16:
            engines.append((rsos.ENGINE_RESIDENT, 0))
        o = oracle_mod.Oracle(L, N, R, seed, tile=S, subsweeps=K, first_real=first)
        o.advance(3)
        for eng, ln in engines:
            g = rsos.Rsos(L, N, R, seed, tile=S, subsweeps=K, first_real=first, engine=eng, lanes=ln)
            g.advance(1)
            g.advance(2)
            compare(g, o, "random L=%d N=%d R=%d S=%d K=%d engine=%d lanes=%d" % (L, N, R, S, K, eng, ln))
            g.close()
        o.close()
        done += 1


def test_largest_lattice_properties(rsos):
    """L = 65536 (the largest the ABI accepts; 2^32 sites, 16 GiB of int32 heights, 1 GiB packed): what holds at any
    size.  sum h = accepted; <h>(t=1) and W^2(t=1) are local quantities, so they must equal the DT(64,1) values of
    the L = 128 ensemble of DESIGN.md section 12 (0.26587, 0.6516) -- here to 4e-4 relative (2^32 sites self-average)."""
    import torch
    free, _ = torch.cuda.mem_get_info()
    if free < 24 * 2 ** 30:
        pytest.skip("needs 24 GiB of device memory")
    g = rsos.Rsos(65536, 1, 1, 7)
    info = g.info()
    assert info["engine"] == "thread" and info["blocks"] == 65536 * 4 * info["lanes"] // 32 * 1
    g.advance(1)
    s1, s2, acc = g.sums()
    assert s1[0] == acc[0] and 0 < acc[0] <= 2 ** 32
    w2, hm = g.width()
    assert abs(w2[0] / 0.265867 - 1) < 4e-4 and abs(hm[0] / (0.65226 * (1 - 0.00101)) - 1) < 4e-4, (w2, hm)
    g.close()


@pytest.mark.parametrize("L,N,R,S,K,mcs,seed", [
    (64, 1, 5, 8, 1, 6, 1),          # the paper's 8 x 8 domains: 16 cells per pass, several realizations per block
    (128, 1, 70, 8, 2, 4, 2),        # 16 realizations per block, ragged last block (70 = 4 * 16 + 6)
    (256, 3, 3, 16, 4, 4, 3),        # 16 x 16 cells, 4-bit sites, K = 4
    (512, 1, 2, 16, 1, 3, 4),        # 128 KiB lattice per block, 2-bit packed lattice spread to nibbles
    (512, 2, 1, 8, 1, 2, 5),         # 1024 cells per pass: one thread each
    (32, 1, 100, 8, 1, 8, 6),        # 4 cells per pass, 100 realizations in one block (400 threads)
    (16, 7, 9, 8, 2, 10, 7),         # one cell per pass; largest N
    (64, 1, 3, 16, 8, 5, 8),         # 32 attempts per cell and pass
])
def test_dt_fine_engine_equals_oracle(rsos, oracle_mod, L, N, R, S, K, mcs, seed):
    """The FINE engine (rsos_fine.cu): DT(c, K) with c = 8 or 16, one thread per cell on a 4-bit lattice resident in
    shared memory for all passes of a call; engine = auto picks it for these shapes."""
    g = rsos.Rsos(L, N, R, seed, tile=S, subsweeps=K, first_real=seed)
    o = oracle_mod.Oracle(L, N, R, seed, tile=S, subsweeps=K, first_real=seed)
    info = g.info()
    assert info["mode"] == "DT" and info["engine"] == "fine" and not info["int32_allocated"], info
    for step in (1, 1, mcs - 2):
        g.advance(step)
        o.advance(step)
        compare(g, o, "DT fine L=%d N=%d S=%d K=%d t=%d" % (L, N, S, K, g.t))
    g.close()


def test_dt_fine_engine_saturated_restart_and_cross_engine(rsos, oracle_mod):
    """FINE engine far from the flat start (L = 64, N = 1, DT(8,1), t = 3000: |h| ~ 900, saturated): snapshot to the
    oracle, both advance; and the THREAD engine run on the same schedule gives the same surface."""
    L, N, R, seed = 64, 1, 6, 13
    g = rsos.Rsos(L, N, R, seed, tile=8)
    assert g.info()["engine"] == "fine"
    g.advance(3000)
    h, (_, _, acc) = g.heights(), g.sums()
    assert h.min() > 500
    o = oracle_mod.Oracle(L, N, R, seed, tile=8)
    o.set_state(h, 3000, acc)
    t = rsos.Rsos(L, N, R, seed, tile=8, engine=rsos.ENGINE_THREAD)
    t.set_state(h, 3000, acc)
    for x in (g, o, t):
        x.advance(3)
    compare(g, o, "fine saturated")
    compare(t, o, "thread on the same cells")
    g.close()
    t.close()


@pytest.mark.parametrize("L,N,R,S,mcs,seed", [(64, 1, 9, 8, 5, 1), (128, 2, 40, 8, 3, 2), (256, 1, 3, 16, 3, 3),
                                              (512, 1, 1, 8, 2, 4), (32, 7, 20, 16, 6, 5)])
def test_dt_fine_engine_poisson_variant_equals_oracle(rsos, oracle_mod, L, N, R, S, mcs, seed):
    """opts.poisson: DTP(c) -- K = c^2 / 4 sub-sweeps per MCS, Poisson(4) attempts per cell and
    sub-sweep from the inversion table; FINE engine against the oracle's DTP, bit for bit."""
    g = rsos.Rsos(L, N, R, seed, tile=S, poisson=True, first_real=3)
    o = oracle_mod.Oracle(L, N, R, seed, tile=S, poisson=True, first_real=3)
    info = g.info()
    assert info["engine"] == "fine" and info["K"] == S * S // 4, info
    for step in (1, mcs - 1):
        g.advance(step)
        o.advance(step)
        compare(g, o, "DTP fine L=%d N=%d S=%d t=%d" % (L, N, S, g.t))
    g.close()
    for kw in (dict(tile=32), dict(tile=8, subsweeps=4), dict(tile=8, engine=rsos.ENGINE_THREAD)):
        with pytest.raises(rsos.RsosError):
            rsos.Rsos(64, 1, 1, 1, poisson=True, **kw)


@pytest.mark.parametrize("L,N,R,mcs,first", [(32, 1, 256, 6, 0), (16, 2, 70, 9, 96), (8, 31, 33, 12, 32), (32, 1, 20, 4, 224)])
def test_multisurface_shared_coordinates_equals_oracle(rsos, oracle_mod, L, N, R, mcs, first):
    """opts.multisurface: the paper's shared-coordinate multisurface scheme (schedule MS) on
    the MULTI engine (realizations innermost in shared memory) against the oracle's MS, bit for bit; R spans several
    groups of 128 and ragged warps."""
    g = rsos.Rsos(L, N, R, 6, multisurface=True, first_real=first)
    o = oracle_mod.Oracle(L, N, R, 6, multisurface=True, first_real=first)
    assert g.info()["engine"] == "multi" and g.info()["mode"] == "RS"
    for step in (1, mcs - 1):
        g.advance(step)
        o.advance(step)
        compare(g, o, "MS L=%d N=%d t=%d" % (L, N, g.t))
    g.close()
    for kw in (dict(first_real=5), dict(tile=8), dict(engine=rsos.ENGINE_ONCHIP)):
        with pytest.raises(rsos.RsosError):
            rsos.Rsos(32, 1, 32, 1, multisurface=True, **kw)
    with pytest.raises(rsos.RsosError):
        rsos.Rsos(64, 1, 32, 1, multisurface=True)


def test_multisurface_long_launch_chunks(rsos, oracle_mod):
    """More than 4096 MCS in one call (the int16 on-chip heights are re-based every 4096 MCS) and a saturated surface."""
    L, N, R = 8, 1, 32
    g = rsos.Rsos(L, N, R, 3, multisurface=True)
    o = oracle_mod.Oracle(L, N, R, 3, multisurface=True)
    g.advance(9000)
    o.advance(9000)
    compare(g, o, "MS 9000 MCS")
    g.close()


@pytest.mark.parametrize("L,N,R,mcs,seed", [(16, 1, 3, 40, 1), (32, 2, 5, 25, 2), (64, 1, 2, 12, 3), (128, 3, 1, 5, 4),
                                            (32, 31, 2, 20, 5), (64, 127, 1, 6, 6)])
def test_rs_level_engine_equals_oracle(rsos, oracle_mod, L, N, R, mcs, seed):
    """The LEVEL engine (rsos_level.cu): serial RS, a block per realization, batches of 256 attempts executed in
    dependency levels -- the sequential result, bit for bit; several MCS per launch; heights far from the flat start."""
    g = rsos.Rsos(L, N, R, seed, tile=L, engine=rsos.ENGINE_LEVEL, first_real=2)
    o = oracle_mod.Oracle(L, N, R, seed, tile=L, first_real=2)
    assert g.info()["engine"] == "level" and g.info()["mode"] == "RS"
    for step in (1, 1, mcs - 2):
        g.advance(step)
        o.advance(step)
        compare(g, o, "RS level L=%d N=%d t=%d" % (L, N, g.t))
    g.advance(700)                                           # |h| beyond one byte: the mod-256 heights wrap
    o.advance(700)
    compare(g, o, "RS level late")
    g.close()


def test_random_shapes_new_engines(rsos, oracle_mod):
    """Seeded random sweep over the engines added in round 2 (FINE and its Poisson variant, LEVEL, general L, MULTI):
    random L, N, R, tile, K, first_real; heights, sums and doubles against the oracle."""
    rng = np.random.default_rng(20261105)
    cases = []
    for _ in range(8):                                                   # FINE
        S = int(rng.choice([8, 16]))
        L = int(rng.choice([l for l in (16, 32, 64, 128, 256) if l >= 2 * S]))
        K = int(rng.choice([k for k in (1, 2, 4, 8) if S * S // k >= 32]))
        cases.append(("fine", dict(L=L, N=int(rng.integers(1, 8)), R=int(rng.integers(1, 40)), tile=S, subsweeps=K)))
    for _ in range(3):                                                   # FINE, Poisson variant
        S = int(rng.choice([8, 16]))
        L = int(rng.choice([l for l in (32, 64, 128) if l >= 2 * S]))
        cases.append(("fine", dict(L=L, N=int(rng.integers(1, 8)), R=int(rng.integers(1, 20)), tile=S, poisson=True)))
    for _ in range(5):                                                   # LEVEL (few realizations, serial RS)
        L = int(rng.choice([16, 32, 64]))
        cases.append(("level", dict(L=L, N=int(rng.integers(1, 12)), R=int(rng.integers(1, 6)), tile=L)))
    for _ in range(8):                                                   # general L: windowed pass, global pass, RSG
        S = int(rng.choice([8, 16, 32]))
        L = int(rng.integers(24, 260))
        while L & (L - 1) == 0:
            L += 1
        K = int(rng.choice([k for k in (1, 2, 4) if S * S // k >= 32]))
        cases.append(("simple", dict(L=L, N=int(rng.integers(1, 10)), R=int(rng.integers(1, 5)), tile=S, subsweeps=K)))
    for _ in range(3):                                                   # MULTI
        L = int(rng.choice([8, 16, 32]))
        cases.append(("multi", dict(L=L, N=int(rng.integers(1, 6)), R=int(rng.integers(1, 150)), multisurface=True,
                                    first_real=32 * int(rng.integers(0, 9)))))
    for want, kw in cases:
        kw = dict(kw)
        kw.setdefault("first_real", int(rng.integers(0, 50)))
        seed = int(rng.integers(1, 1 << 40))
        mcs = int(rng.integers(2, 5))
        L, N, R = kw.pop("L"), kw.pop("N"), kw.pop("R")
        g = rsos.Rsos(L, N, R, seed, **kw)
        o = oracle_mod.Oracle(L, N, R, seed, **kw)
        assert g.info()["engine"] == want, (want, L, N, R, kw, g.info())
        g.advance(mcs)
        o.advance(mcs)
        compare(g, o, "%s L=%d N=%d R=%d %s" % (want, L, N, R, kw))
        g.close()
        o.close()
