"""Pins for the oracle's Philox4x32-10 (BASELINE.json north_star (1))."""
import os
import shutil
import subprocess

import numpy as np
import pytest

HERE = os.path.dirname(os.path.abspath(__file__))


def test_philox_known_answers(oracle_mod):
    rows = [l.split() for l in open(os.path.join(HERE, "golden", "philox_kat.txt")) if l.strip() and l[0] != "#"]
    assert len(rows) == 3
    for r in rows:
        v = [int(x, 16) for x in r]
        out = oracle_mod.philox(v[0:4], v[4:6])
        assert [int(x) for x in out] == v[6:10]


def test_philox_bijective_per_key(oracle_mod):
    # distinct counters -> distinct outputs under one key (Philox is a keyed bijection)
    key = (123456789, 987654321)
    seen = set()
    for q in range(64):
        for tile in range(8):
            for u in range(8):
                seen.add(tuple(int(x) for x in oracle_mod.philox((q, tile, u, 5), key)))
    assert len(seen) == 64 * 8 * 8


def test_philox_each_word_sensitive(oracle_mod):
    # changing any one counter or key word changes the output (catches a dropped operand)
    base_c, base_k = [1, 2, 3, 4], [5, 6]
    ref = oracle_mod.philox(base_c, base_k)
    for i in range(4):
        c = list(base_c); c[i] ^= 0x10000
        assert (oracle_mod.philox(c, base_k) != ref).any()
    for i in range(2):
        k = list(base_k); k[i] ^= 0x10000
        assert (oracle_mod.philox(base_c, k) != ref).any()


@pytest.mark.skipif(shutil.which("nvcc") is None, reason="nvcc needed to compile the cuRAND header helper")
def test_philox_matches_curand_header(oracle_mod, tmp_path):
    exe = str(tmp_path / "curand_philox_host")
    subprocess.check_call(["nvcc", "-O1", "-o", exe, os.path.join(HERE, "curand_philox_host.cu")])
    n = 20000
    out = subprocess.check_output([exe, str(n), "42"]).decode().split("\n")
    rows = [[int(x, 16) for x in l.split()] for l in out if l.strip()]
    assert len(rows) == n
    for v in rows:
        got = oracle_mod.philox(v[0:4], v[4:6])
        assert [int(x) for x in got] == v[6:10]
