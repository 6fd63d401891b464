"""Host-side pieces of bench.py (no GPU): every leg of the default run names a valid workload, and the instruction
roofline is the number DESIGN.md section 6 derives (profiles/r2_sass_attempt_loop.md)."""
import importlib.util
import os

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def bench():
    spec = importlib.util.spec_from_file_location("bench_mod", os.path.join(ROOT, "bench.py"))
    m = importlib.util.module_from_spec(spec)
    spec.loader.exec_module(m)
    return m


def test_legs_resolve(bench):
    import paper_1605_02620_b200 as pkg
    from paper_1605_02620_b200.utils import workloads
    assert bench.EXTRA_LEGS[0] == "C4"                       # the other north_star config comes first
    for name in ("C2",) + bench.EXTRA_LEGS:
        c = bench.leg_config(name)
        assert c["mcs_per_step"] >= 1 and c["R"] * c["L"] ** 2 >= 1 << 17
        pl = pkg.plan(c["L"], c["N"], c["R"], tile=c["tile"], subsweeps=c["subsweeps"])   # host-only: needs no device
        assert pl["engine"] in ("thread", "resident", "onchip", "level"), (name, pl)
    assert bench.leg_config("C5/L=256")["R"] == workloads.c5_realizations(256) == 256
    assert bench.leg_config("C3/N=2")["N"] == 2


def test_alu_peak_is_the_documented_one(bench):
    # 148 SMs x 4 x 32 / 52.25 cycles per 32 attempts x 1.965 GHz = 712 G attempts/s
    assert bench.alu_peak_attempts_per_s(148, 1965.0) == pytest.approx(712.4e9, rel=1e-3)
    assert 2 * bench.IDEAL_LOOP["alu_pipe"] == pytest.approx(52.25)
