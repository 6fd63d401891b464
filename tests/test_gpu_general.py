"""GPU parity for lattice sides that are not powers of two (S 8(f) NEXT-3): the general-L
schedule RSG / DTG through the C ABI against the CPU oracle, bit-exact (heights, S1, S2, accepted, W2 / <h>
doubles, power sums), including the paper's largest system L = 9605 for a prefix."""
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


def _same(g, o, R):
    for a, b in zip(g.sums(), o.sums()):
        assert (a == b).all()
    gw, gh = g.width()
    ow, oh = o.width()
    assert (gw == ow).all() and (gh == oh).all()
    assert np.array_equal(g.heights(), o.heights())


@pytest.mark.parametrize("L,N,R,S,K,mcs,first", [
    (150, 1, 3, 64, 1, 5, 0),        # DTG, T = 2, four tiles of 75 x 75
    (200, 2, 2, 32, 4, 4, 5),        # DTG, T = 6, widths 33 / 34, four sub-sweeps of unequal attempt counts
    (100, 1, 2, 8, 2, 3, 0),         # DTG, T = 12
    (333, 3, 1, 16, 1, 2, 1),        # DTG, T = 20, odd L: scalar reductions
    (150, 9, 2, 64, 1, 3, 0),        # N > 7: thread per tile in global memory (the windowed kernel needs N <= 7)
    (1000, 7, 35, 64, 2, 2, 3),      # T = 14: 49 tiles per pass and realization, ragged last warp of 16 tiles, N = 7
    (300, 1, 2, 128, 1, 2, 0),       # T = 2, tiles of 150 x 150: windows too large for shared memory -> global path
    (220, 1, 2, 64, 1, 3, 0),        # T = 2, tiles of 110 x 110: the widest windows the shared-memory kernel takes
    (255, 2, 2, 64, 1, 3, 1),        # T = 2, tiles of 127 / 128: window rows of 130 columns exceed the 128 the kernel stages
    (45, 1, 4, 64, 1, 12, 0),        # RSG (2S > L), odd L
    (6, 1, 5, 64, 1, 40, 2),         # RSG, tiny
])
def test_general_lattice_equals_oracle(rsos, oracle_mod, L, N, R, S, K, mcs, first):
    g = rsos.Rsos(L, N, R, 3, tile=S, subsweeps=K, first_real=first)
    o = oracle_mod.Oracle(L, N, R, 3, tile=S, subsweeps=K, first_real=first)
    info = g.info()
    assert info["engine"] == "simple" and info["mode"] == o.mode
    for step in (1, mcs - 1):
        g.advance(step)
        o.advance(step)
        _same(g, o, R)
    base, M = g.moments()
    for r in range(R):
        assert M[r] == o.power_sums(r, int(base[r]))
    g.close()
    o.close()


@pytest.mark.parametrize("L,N,R,K,mcs,first", [
    (130, 1, 3, 1, 6, 0),            # T = 2: four tiles of 65 x 65, every tile wraps around the lattice edge sooner or later
    (131, 2, 2, 2, 5, 4),            # tiles of 65 / 66 sites, 4-bit sites, two sub-sweeps of unequal attempt counts
    (132, 7, 1, 1, 4, 0),            # 66 x 66 tiles (the largest the window takes), largest N
    (263, 1, 40, 4, 3, 2),           # T = 4: 160 tiles per pass = 5 warps, K = 4
    (260, 3, 2, 1, 4, 0),            # L * FB is a multiple of 32 (no partial last word), 4-bit sites
    (1290, 1, 1, 1, 2, 0),           # T = 20: 100 tiles per pass, rows of 81 packed words
])
def test_general_lattice_packed_engine_equals_oracle(rsos, oracle_mod, L, N, R, K, mcs, first):
    """General L on the PACKED lattice (rsos_gthread.cu; tile 64, N <= 7, ceil(L / T) <= 66): lane per tile with bit-range
    staging / write-back across the periodic row end; sums straight from the packed lattice at every step, heights and
    moments through the rebuild, all against the oracle's DTG."""
    g = rsos.Rsos(L, N, R, 5, subsweeps=K, first_real=first)
    o = oracle_mod.Oracle(L, N, R, 5, subsweeps=K, first_real=first)
    info = g.info()
    assert info["engine"] == "thread" and info["lanes"] == 1 and info["packed_bits"] == (2 if N == 1 else 4), info
    assert not info["int32_allocated"]
    for step in (1,) * (mcs - 1):
        g.advance(step)
        o.advance(step)
        for a, b in zip(g.sums(), o.sums()):                 # packed sums, no int32 rebuild
            assert (a == b).all()
    assert not g.info()["int32_allocated"]
    g.advance(1)
    o.advance(1)
    _same(g, o, R)
    base, M = g.moments()
    for r in range(R):
        assert M[r] == o.power_sums(r, int(base[r]))
    # snapshot restart through the packed state, and the SIMPLE engine on the same schedule
    snap, (_, _, acc) = g.heights(), g.sums()
    s2 = rsos.Rsos(L, N, R, 5, subsweeps=K, first_real=first, engine=rsos.ENGINE_SIMPLE)
    s2.set_state(snap, g.t, acc)
    g.set_state(snap, g.t, acc)
    for x in (g, s2, o):
        x.advance(2)
    _same(g, o, R)
    _same(s2, o, R)
    g.close()
    s2.close()
    o.close()


def test_general_lattice_snapshot_restart(rsos, oracle_mod):
    """set_state / get_heights on a general lattice: the oracle continues from a GPU snapshot (t enters the counter)."""
    L, N, R = 150, 1, 2
    g = rsos.Rsos(L, N, R, 8)
    g.advance(7)
    snap, (_, _, acc) = g.heights(), g.sums()
    o = oracle_mod.Oracle(L, N, R, 8)
    o.set_state(snap, 7, acc)
    g.advance(3)
    o.advance(3)
    _same(g, o, R)
    g2 = rsos.Rsos(L, N, R, 8)
    g2.set_state(snap, 7, acc)
    g2.advance(3)
    _same(g2, o, R)
    bad = snap.copy()
    bad[0, 0, 0] += 5
    with pytest.raises(rsos.RsosError) as e:
        g2.set_state(bad, 7, acc)
    assert e.value.code == rsos.binding.RSOS_EINVAL
    for x in (g, g2):
        x.close()
    o.close()


def test_general_lattice_refuses_other_engines(rsos):
    for eng in (rsos.ENGINE_THREAD, rsos.ENGINE_WARP, rsos.ENGINE_RESIDENT, rsos.ENGINE_ONCHIP):   # 75-site tiles: no THREAD
        with pytest.raises(rsos.RsosError) as e:
            rsos.Rsos(150, 1, 1, 1, engine=eng)
        assert e.value.code == rsos.binding.RSOS_EUNSUP


@pytest.mark.parametrize("engine", ["auto", "simple"])
def test_paper_largest_system_prefix(rsos, oracle_mod, engine):
    """L = 9605 ('bounded by memory constraints'), N = 1, one realization, DTG(64,1): 150 x 150 tiles of 64 / 65
    sites, 5625 per colour pass; 2 MCS = 1.8e8 attempts, every height compared with the oracle.  engine = auto is the
    lane-per-tile engine on the packed lattice (23 MiB instead of 369 MiB), simple the byte-window path on int32."""
    L = 9605
    g = rsos.Rsos(L, 1, 1, 1, engine=rsos.ENGINE_AUTO if engine == "auto" else rsos.ENGINE_SIMPLE)
    assert g.info()["engine"] == ("thread" if engine == "auto" else "simple")
    o = oracle_mod.Oracle(L, 1, 1, 1)
    g.advance(2)
    o.advance(2)
    _same(g, o, 1)
    W2, hm = g.width()
    assert 0.3 < W2[0] < 0.4 and 1.0 < hm[0] < 1.2           # W^2(2) = 0.339 on a large lattice (C2 time series)
    g.close()
    o.close()
