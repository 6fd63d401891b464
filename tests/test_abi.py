"""CPU-side checks of the boundary: librsos.so builds (nvcc cross-compiles for sm_100a), loads, and
exports exactly the entry points include/rsos.h declares; without a GPU every call fails loudly
(no CPU fallback); the product package never imports the oracle."""
import ctypes
import os
import re
import subprocess

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def lib_path():
    from paper_1605_02620_b200 import build
    return build.build()


def header_functions():
    src = open(os.path.join(ROOT, "include", "rsos.h")).read()
    src = re.sub(r"/\*.*?\*/", "", src, flags=re.S)
    return sorted(set(re.findall(r"\b(rsos_[a-z_]+)\s*\(", src)))


def test_header_declares_the_north_star_calls():
    names = header_functions()
    for need in ("rsos_init", "rsos_advance", "rsos_width"):
        assert need in names


def test_library_exports_every_declared_symbol(lib_path):
    import paper_1605_02620_b200 as m
    names = header_functions()
    assert sorted(m.SYMBOLS) == names
    out = subprocess.check_output(["nm", "-D", "--defined-only", lib_path], text=True)
    exported = sorted(set(re.findall(r" T (rsos_[a-z_]+)$", out, flags=re.M)))
    assert exported == names
    lib = ctypes.CDLL(lib_path)
    for n in names:
        assert getattr(lib, n) is not None


def test_library_is_sm100a_only(lib_path):
    out = subprocess.check_output(["cuobjdump", "-lelf", lib_path], text=True)
    archs = set(re.findall(r"sm_(\d+a?)", out))
    assert archs == {"100a"}, archs


def test_no_cpu_fallback_without_a_device():
    import torch
    if torch.cuda.is_available():
        pytest.skip("a CUDA device is present")
    import paper_1605_02620_b200 as m
    with pytest.raises(m.RsosError) as e:
        m.Rsos(32, 1, 4, 1)
    assert e.value.code == -4
    with pytest.raises(m.RsosError):
        m.philox([[0, 0, 0, 0]], [[0, 0]])


def test_argument_errors_need_no_device(lib_path):
    import paper_1605_02620_b200 as m
    for args, kw, code in [((3, 1, 1, 1), {}, -1), ((70000, 1, 1, 1), {}, -1), ((48, 1, 1, 1), dict(engine=m.ENGINE_ONCHIP), -5),
                           ((150, 1, 1, 1), dict(engine=m.ENGINE_THREAD), -5), ((64, 0, 1, 1), {}, -1), ((64, 1, 0, 1), {}, -1),
                           ((128, 1, 1, 1), dict(tile=24), -1), ((64, 1, 1, 1), dict(engine=m.ENGINE_WARP), -5),
                           ((256, 1, 1, 1), dict(engine=m.ENGINE_ONCHIP), -5), ((128, 32, 1, 1), dict(engine=m.ENGINE_WARP), -5),
                           ((128, 1, 1, 1), dict(lanes=3), -1), ((128, 8, 1, 1), dict(engine=m.ENGINE_THREAD), -5),
                           ((256, 1, 1, 1), dict(engine=m.ENGINE_THREAD, tile=128), -5)]:
        with pytest.raises(m.RsosError) as e:
            m.Rsos(*args, **kw)
        assert e.value.code == code, (args, kw)


def test_product_never_touches_the_oracle():
    pkg = os.path.join(ROOT, "paper_1605_02620_b200")
    for dirpath, _, files in os.walk(pkg):
        for f in files:
            if f.endswith((".py", ".cu", ".cuh", ".h")):
                text = open(os.path.join(dirpath, f)).read()
                assert not re.search(r"^\s*(from|import)\s+oracle|rsos_oracle|#include\s+\".*oracle", text, flags=re.M), f
    for f in os.listdir(os.path.join(ROOT, "oracle")):
        if f.endswith((".py", ".c")):
            text = open(os.path.join(ROOT, "oracle", f)).read()
            assert not re.search(r"^\s*(from|import)\s+paper_1605_02620_b200|#include\s+\".*csrc", text, flags=re.M), f


def test_plan_picks_engines_lanes_and_site_width(lib_path):
    """rsos_plan: the host-side selection logic of rsos_init, no device needed."""
    import paper_1605_02620_b200 as m
    from paper_1605_02620_b200.utils import workloads as w
    c = w.CONFIGS
    p = m.plan(c["C1"]["L"], 1, c["C1"]["R"])
    assert (p["mode"], p["engine"], p["S"], p["K"], p["launches_per_mcs"]) == ("RS", "level", 32, 1, 1)   # 128 chains: few realizations
    assert m.plan(32, 1, 4096)["engine"] == "onchip"                                  # many realizations: a warp each
    p = m.plan(c["C2"]["L"], 1, c["C2"]["R"])
    assert (p["mode"], p["engine"], p["pass_tiles"], p["lanes"], p["packed_bits"]) == ("DT", "thread", 8192, 4, 2)
    p = m.plan(c["C3"]["L"], 1, c["C3"]["R"])
    assert (p["engine"], p["pass_tiles"], p["lanes"], p["packed_bits"]) == ("thread", 16384, 2, 2)
    p = m.plan(c["C3"]["L"], 4, c["C3"]["R"])
    assert (p["engine"], p["lanes"], p["packed_bits"]) == ("thread", 4, 4)         # 4-bit sites for N = 2..7
    p = m.plan(c["C4"]["L"], 1, 1)
    assert (p["engine"], p["pass_tiles"], p["lanes"], p["launches_per_mcs"]) == ("thread", 65536, 2, 4)
    for L, cl in ((128, 1), (256, 1), (512, 2)):                                      # C5: few tiles per pass -> lattice on chip
        for N in (1, 2):
            p = m.plan(L, N, w.c5_realizations(L), tile=64, subsweeps=4)
            assert (p["engine"], p["pass_tiles"], p["launches_per_mcs"], p["cluster"], p["lanes"], p["packed_bits"]) == \
                ("resident", 1024, 1, cl, 32, 2 * N), (L, N, p)
    assert m.plan(512, 1, 64, tile=64, subsweeps=4, cluster=8)["cluster"] == 8        # any cluster size that divides the 16 tiles
    with pytest.raises(m.RsosError) as e:
        m.plan(512, 1, 64, tile=64, subsweeps=4, engine=m.ENGINE_RESIDENT, cluster=1) # 256 KiB of uint8 sites do not
    assert e.value.code == -5
    p = m.plan(128, 1, 1024, tile=64, subsweeps=4, engine=m.ENGINE_WARP)
    assert (p["engine"], p["launches_per_mcs"]) == ("warp", 16)
    assert m.plan(2048, 1, 1)["engine"] == "warp"                                    # 256 tiles per pass: not resident, too few for THREAD
    assert m.plan(64, 1, 4096)["engine"] == "onchip" and m.plan(512, 1, 2, tile=512)["engine"] == "simple"
    assert m.plan(256, 8, 4096)["engine"] == "warp" and m.plan(256, 40, 4096)["engine"] == "simple"
    assert m.plan(1024, 1, 128, tile=8)["packed_bits"] == 4                          # 8 < 16 sites per 2-bit word
    assert m.plan(1024, 1, 128, subsweeps=128)["lanes"] == 4                         # 32 attempts per tile: 8 * 4 fits
    assert m.plan(1024, 1, 128, subsweeps=128, engine=m.ENGINE_THREAD, lanes=2)["lanes"] == 2
    with pytest.raises(m.RsosError) as e:
        m.plan(1024, 1, 128, subsweeps=128, engine=m.ENGINE_THREAD, lanes=8)         # a batch of 64 attempts does not fit
    assert e.value.code == -1
    # lattice sides that are not powers of two: the general-L schedule, SIMPLE engine
    p = m.plan(9605, 1, 128)                      # tiles of 64 / 65 sites fit the packed windows: lane-per-tile engine
    assert (p["mode"], p["engine"], p["S"], p["pass_tiles"], p["lanes"], p["packed_bits"]) == ("DT", "thread", 64, 128 * 75 * 75, 1, 2)
    assert m.plan(9605, 9, 1)["engine"] == "simple" and m.plan(150, 1, 4)["engine"] == "simple"   # N > 7; 75-site tiles
    p = m.plan(100, 1, 4)
    assert (p["mode"], p["engine"], p["S"]) == ("RS", "simple", 100)
    # fewer SMs: the same pass reaches six warps per SM with fewer lanes
    assert m.plan(c["C2"]["L"], 1, c["C2"]["R"], sm_count=16)["lanes"] == 2
