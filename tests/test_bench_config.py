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
    assert bench.EXTRA_LEGS[0] == "C4" and bench.DEFAULT_LEGS == ("C4",)   # the other north_star config comes first
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


def fake_leg(bench, name, engine):
    """A run_leg record with every field filled with long, realistic values (no GPU)."""
    c = bench.leg_config(name)
    info = {"mode": "DT", "engine": engine, "S": 64, "K": 1, "launches": 123456, "sm_count": 148, "smem_bytes": 227 * 1024,
            "blocks": 1024, "lanes": 4, "packed_bits": 2, "cluster": 0, "int32_allocated": True}
    peak, src = bench.engine_peak(info, 1965.0)
    return {"workload": name, "value": 198.76543210987, "unit": bench.UNIT, "steps": 20, "warmup": 3, "reps": 3,
            "region_ms": [434.123456, 435.123456, 436.123456], "ms_per_step": 21.7561234567,
            "config": bench.config_dict_for(name, c, 8), "residency": bench.l2_note(c, info), "engine": info,
            "clocks": {"sm_mhz": 1965.0, "sm_max_mhz": 1965.0, "reasons": ["sw_power_cap", "sw_thermal_slowdown"], "power_w_max": 987.65, "samples": 27},
            "e2e": {"value": 132.123456789, "unit": bench.UNIT, "h2d_bytes_per_step": 536871936, "d2h_bytes_per_step": 5124, "what": "x" * 90},
            "gpu_launches": 2581,
            "roofline": {"bound": "alu" if peak else "latency", "achieved": 199.123456789, "peak": peak / 1e9 if peak else None,
                         "unit": bench.UNIT, "frac": 0.279123456 if peak else None, "traffic": 17301234.0, "traffic_source": "y" * 80,
                         "peak_source": src, "kernel": "update kernel, engine=thread", "attempts_per_launch": 33554432.0,
                         "avg_launch_ms": 0.168812345, "update_launches": 7680, "update_share_of_step": 0.99312345,
                         "frac_of_survey_floor_22_instr": 0.11712345,
                         "int32_equiv_sweep": {"bytes_per_attempt": 8.25, "GBps": 1640.123456, "hbm_peak_GBps": 6540.8,
                                               "peak_source": "measured (MEASURED_PEAKS.json hbm_gbs)", "frac": 0.25112345}},
            "result_check": {"W2_mean": 1.23456789012, "hmean_mean": 187.123456789, "t_mcs": 2048}}


def test_final_line_is_small_and_complete(bench):
    """The driver keeps only a few KB of bench.py's output (round 2's 21 KB line was cut and left the round without a parsed
    record): the final line must stay below 2 KB with every side number present, and carry the contract's keys."""
    import json
    c = bench.leg_config("C2")
    head, c4 = fake_leg(bench, "C2", "thread"), fake_leg(bench, "C4", "thread")
    cpu = {"value": 0.759123456, "unit": bench.UNIT, "cores": 16, "kind": "oracle",
           "sample": "16 of 128 realizations, L=1024, 1234 MCS per step x 1 step(s) + width, OpenMP threads=16",
           "c1_full_1thread": 0.04512345, "c4_cut_2mcs_allcores": 0.7123456}
    s4 = {"value": 287.123456, "ms_per_step": 59.8123456, "what": "z" * 60}
    line = bench.make_line(c, 8, 20, 3, head, cpu, c4, s4, "/root/repo/bench_legs.json")
    text = json.dumps(line)
    assert len(text) < bench.MAX_LINE_BYTES == 2048, len(text)
    for k in ("metric", "value", "unit", "n_gpus", "steps", "warmup", "ms_per_step", "higher_is_better", "scaling", "vs_baseline",
              "dtype", "data", "config", "clocks", "e2e", "gpu_launches", "roofline", "cpu_baseline", "c4", "c2_seeds4"):
        assert k in line, k
    assert set(line["roofline"]) >= {"bound", "achieved", "peak", "unit", "frac", "traffic", "frac_hbm_int32_equiv",
                                    "frac_of_survey_floor_22_instr", "avg_launch_ms", "attempts_per_launch"}
    assert set(line["e2e"]) == {"value", "unit", "h2d_bytes_per_step", "d2h_bytes_per_step"}
    assert set(line["cpu_baseline"]) >= {"value", "unit", "cores", "kind", "sample"}
    assert "model" not in line["config"] and line["config"]["workload"].startswith("C2")


def test_config_is_the_same_for_both_arms(bench):
    """`config` must not depend on the engine: the driver compares the two arms' config objects."""
    c = bench.leg_config("C2")
    a = bench.config_dict_for("C2", c, 1, {"engine": "thread", "packed_bits": 2})
    b = bench.config_dict_for("C2", c, 1, None)
    assert a == b


def test_no_instruction_peak_is_claimed_for_other_engines(bench):
    """The SASS count behind the alu peak is the THREAD engine's loop; LEVEL, RESIDENT, ... report frac = null."""
    for eng in ("level", "resident", "fine", "onchip", "warp", "simple", "multi"):
        peak, src = bench.engine_peak({"engine": eng, "sm_count": 148}, 1965.0)
        assert peak is None and eng in src
    peak, _ = bench.engine_peak({"engine": "thread", "sm_count": 148}, 1965.0)
    assert peak == pytest.approx(712.4e9, rel=1e-3)


def test_selfcheck_cases_resolve_to_their_engines():
    """paper_1605_02620_b200.selfcheck: every case of the engine tour selects the engine it names (host-only planning)."""
    import paper_1605_02620_b200 as pkg
    from paper_1605_02620_b200 import selfcheck
    seen = set()
    for name, L, N, R, kw, engine in selfcheck.CASES:
        pl = pkg.plan(L, N, R, **kw)
        assert pl["engine"] == engine, (name, pl)
        if "lanes" in kw:
            assert pl["lanes"] == kw["lanes"], name
        if "cluster" in kw:
            assert pl["cluster"] == kw["cluster"], name
        seen.add(engine)
    assert seen == {"thread", "resident", "fine", "level", "onchip", "multi", "warp", "simple"}
