#!/usr/bin/env python
"""bench.py -- RSOS site-update attempts per second on B200 (BASELINE.json metric), one JSON line.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--workload C2|C4|C3/N=2|C5/L=256|...] [--impl reference]

A *step* is one pass of the whole hot path over one
batch: `mcs_per_step` Monte-Carlo steps of rsos_advance (Philox draws, origin draw, tile staging,
attempt loop, write-back) followed by one rsos_width (int64 width reduction, result read to host).
The headline workload is BASELINE.json configs[1] (C2: L=1024, N=1, 128 realizations, DT(64,1)), seed 1.

Output.  The LAST stdout line is ONE compact JSON object (< 2 KB, checked before printing: the driver keeps only a few
KB of output) that carries the C2 headline alone, plus two small side numbers: "c4" (the other north_star config,
L=2^15, one surface) and "c2_seeds4" (configs[1] as BASELINE.json words it, "seeds 1..4": four contexts on four
streams, so a colour pass has 32768 tiles in flight instead of 8192).  Everything else -- the full record of every leg
with engine info, clocks and per-kernel numbers, and with --all-legs the legs on C3, C5 and C1 -- is written to the
side file bench_legs.json (git-ignored) and never printed.  Nothing is flushed between steps: a step sweeps the same
resident lattice 4K * mcs_per_step times exactly as a production run does; `config.l2` says so.

`value` is the MEDIAN of --reps (default 3) timed regions of exactly --steps steps each (median of at least
three timed runs); `ms_per_step` belongs to that median region.

value     whole-job attempts/s with the lattice resident on the device (device-timed with CUDA events
          on the stream the kernels run on, barrier + synchronize on both sides, max over ranks).
e2e       the same metric through the C ABI with HOST buffers: every step restores the lattice from
          a pinned host snapshot (rsos_set_state, H2D), advances it, and reads W2/<h> back (D2H).
roofline  dominant kernel (the update kernel), bound "alu": attempts/s of the update launches alone
          (CUDA events inside the library, rsos_kernel_time) against the rate at which the SASS-counted
          ideal attempt loop saturates the integer alu pipe at the SM clock measured during the run
          (DESIGN.md section 6).  `int32_equiv_sweep` keeps north_star's other candidate -- 8.25 B per
          attempt as if the lattice were int32 -- as a labelled equivalent rate; `traffic` is the DRAM
          bytes per launch ncu measured.
cpu_baseline / --impl reference: the CPU oracle as it stands, on a bounded sample of the workload; cpu_baseline also
          carries the two other oracle timings SURVEY 8(d) lists: C1 in full on one thread and a cut-down C4
          (L=32768, 2 MCS) on all cores.
N > 1: replicas only: rank i runs realizations [i*R, (i+1)*R), no collective
on the data path; scaling is weak; the side legs are skipped.
"""
import argparse
import json
import os
import subprocess
import sys
import threading
import time

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

from paper_1605_02620_b200.utils import workloads  # noqa: E402  (no method arithmetic in there)

METRIC = "rsos_site_update_attempts_per_second"
UNIT = "G attempts/s"
BYTES_PER_ATTEMPT = 8.25      # 4 B read + 4 B write per site + (4S+4)/S^2 halo re-read, S = 64
FALLBACK_HBM_GBS = 6650.0     # /opt/skills/guides/B200_PROFILING.md fallback when MEASURED_PEAKS.json is absent


def parse():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=20)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="b200", choices=["b200", "reference"])
    ap.add_argument("--workload", default="C2", help="C1..C5, or e.g. C3/N=2, C5/L=256")
    ap.add_argument("--mcs-per-step", type=int, default=0, help="MCS per step (0 = workload default)")
    ap.add_argument("--engine", default="auto", choices=["auto", "simple", "warp", "onchip", "thread", "resident", "fine", "level"])
    ap.add_argument("--lanes", type=int, default=0, help="THREAD engine lanes per tile (0 = auto)")
    ap.add_argument("--tile", type=int, default=0)
    ap.add_argument("--subsweeps", type=int, default=0)
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-e2e", action="store_true")
    ap.add_argument("--no-extra", action="store_true", help="skip the side legs (C4, C2 with seeds 1..4)")
    ap.add_argument("--all-legs", action="store_true", help="also time C3, C3/N=2, C5 (L=64..512), C1 and X1 (side file only)")
    ap.add_argument("--extra-steps", type=int, default=15, help="timed steps of each side leg (15: >= 10 clock samples per leg)")
    ap.add_argument("--reps", type=int, default=3, help="timed regions of --steps steps each; the median is reported")
    ap.add_argument("--legs-file", default=os.path.join(ROOT, "bench_legs.json"), help="where the full per-leg records go")
    ap.add_argument("--cpu-seconds", type=float, default=12.0, help="target CPU time of the oracle sample")
    return ap.parse_args()


# side legs: the default run times the other north_star config (C4); --all-legs adds the rest (side file only)
DEFAULT_LEGS = ("C4",)
EXTRA_LEGS = ("C4", "C2", "C3", "C3/N=2", "C5", "C5/L=128", "C5/L=256", "C5/L=512", "C1", "X1")
MAX_LINE_BYTES = 2048         # the driver keeps a few KB of output: the final line must fit whole


def workload(args):
    c = leg_config(args.workload)
    if args.tile:
        c["tile"] = args.tile
    if args.subsweeps:
        c["subsweeps"] = args.subsweeps
    if args.mcs_per_step:
        c["mcs_per_step"] = args.mcs_per_step
    return c


def cpu_model():
    try:
        with open("/proc/cpuinfo") as f:
            for line in f:
                if line.lower().startswith("model name"):
                    return line.split(":", 1)[1].strip()
    except OSError:
        pass
    return "unknown"


def l2_note(c, info):
    """Engine-dependent residency note (full leg record only; `config` must be the same string for both arms)."""
    int32_mib = c["R"] * c["L"] ** 2 * 4 / 2 ** 20
    if info and info.get("engine") in ("resident", "fine", "onchip", "level", "multi"):
        return "lattice in shared memory for all %d MCS of a step; int32 view %.0f MiB" % (c["mcs_per_step"], int32_mib)
    if info and info.get("packed_bits"):
        work = int32_mib * info["packed_bits"] / 32
        return "working lattice %.0f MiB (%d bits/site; int32 view %.0f MiB) vs 126 MB L2: %s" % (
            work, info["packed_bits"], int32_mib, "larger than L2" if work * 2 ** 20 > 126e6 else "L2-resident")
    return "state %.0f MiB int32 vs 126 MB L2" % int32_mib


L2_RULE = "no flush: sweeps revisit the resident lattice as in production (DESIGN.md 6)"


def traffic_note(workload_name, info):
    """(DRAM bytes per launch of the dominant kernel, where it comes from) from the committed ncu --set full
    summaries (profiles/traffic.csv: key, bytes, commit the capture was taken at, capture file), or (None, None)."""
    key = "%s/%s/lanes%d" % (workload_name, info["engine"], info.get("lanes", 0))
    try:
        with open(os.path.join(ROOT, "profiles", "traffic.csv")) as f:
            for line in f:
                parts = line.strip().split(",")
                if len(parts) >= 2 and parts[0] == key:
                    src = "profiles/traffic.csv" + (" (captured at commit %s, %s)" % (parts[2], parts[3]) if len(parts) >= 4 else "")
                    return float(parts[1]), src
    except (OSError, ValueError):
        pass
    return None, None


def config_dict(args, c, n_gpus, info=None):
    return config_dict_for(args.workload, c, n_gpus, info)


def config_dict_for(name, c, n_gpus, info=None):
    mode = "RS" if 2 * c["tile"] > c["L"] else "DT(%d,%d)" % (c["tile"], c["subsweeps"])
    return {"workload": "%s: RSOS N=%d, L=%d periodic, %d realizations per GPU, flat start, seed %d"
                        % (name, c["N"], c["L"], c["R"], c["seed"]),
            "schedule": mode, "mcs_per_step": c["mcs_per_step"],
            "step": "rsos_advance(mcs_per_step) + rsos_width",
            "l2": L2_RULE,
            "parallelism": "replicas x%d, no collective" % n_gpus}


class ClockSampler(threading.Thread):
    """nvidia-smi clocks / throttle reasons during the timed region (B200_PROFILING.md recipe):
    one `nvidia-smi -lms 50` child, rows kept only between mark() and stop()."""
    Q = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,clocks_event_reasons.hw_thermal_slowdown,"
         "clocks_event_reasons.sw_thermal_slowdown,clocks_event_reasons.sw_power_cap")

    def __init__(self, index):
        super().__init__(daemon=True)
        self.rows, self.keep, self.proc = [], False, None
        try:
            self.proc = subprocess.Popen(["nvidia-smi", "-i", str(index), "--query-gpu=" + self.Q,
                                          "--format=csv,noheader,nounits", "-lms", "50"],
                                         stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
        except OSError:
            pass

    def run(self):
        if not self.proc:
            return
        for line in self.proc.stdout:
            f = [x.strip() for x in line.strip().split(",")]
            if self.keep and len(f) >= 7:
                self.rows.append(f)

    def mark(self):
        self.keep = True

    def stop(self):
        self.keep = False
        if self.proc:
            self.proc.terminate()
            try:
                self.proc.wait(timeout=5)
            except subprocess.TimeoutExpired:
                self.proc.kill()
        self.join(timeout=5)
        rows = []
        for r in self.rows:
            try:
                rows.append((float(r[0]), float(r[1]), float(r[2]), r[3:7]))
            except ValueError:
                pass
        if not rows:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["unavailable"], "samples": 0}
        sm = sorted(r[0] for r in rows)
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        reasons = [n for i, n in enumerate(names) if any(r[3][i].lower().startswith("active") for r in rows)]
        return {"sm_mhz": sm[len(sm) // 2], "sm_max_mhz": rows[0][1], "reasons": reasons,
                "power_w_max": max(r[2] for r in rows), "samples": len(rows)}


def peaks():
    path = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(path):
        with open(path) as f:
            return float(json.load(f)["hbm_gbs"]), "measured (MEASURED_PEAKS.json hbm_gbs)"
    return FALLBACK_HBM_GBS, "fallback (B200_PROFILING.md)"


# ---------------------------------------------------------------------------------------------
# CPU oracle legs (the only places bench.py executes oracle/): cpu_baseline and --impl reference
# ---------------------------------------------------------------------------------------------
def oracle_sample(c, seconds, steps=1, warmup=0):
    """Time the oracle as it stands on a bounded sample of workload c: min(R, cores) realizations of
    the same L, N, S, K, for as many MCS as fit in `seconds` of wall time (calibrated on 1 MCS).
    Returns (attempts/s, cores, description, ms per step)."""
    from oracle import rsos_oracle
    rsos_oracle.build()
    cores = os.cpu_count() or 1
    R = min(c["R"], cores)
    o = rsos_oracle.Oracle(c["L"], c["N"], R, c["seed"], tile=c["tile"], subsweeps=c["subsweeps"])
    threads = o.threads
    t0 = time.perf_counter()
    o.advance(1)
    dt1 = max(time.perf_counter() - t0, 1e-4)
    n_total = max(1, steps + warmup)
    mcs = max(1, min(c["mcs_per_step"] if steps > 1 else 10 ** 9, int(seconds / n_total / dt1)))
    for _ in range(warmup):
        o.advance(mcs)
        o.width()
    t0 = time.perf_counter()
    for _ in range(steps):
        o.advance(mcs)
        o.width()
    dt = time.perf_counter() - t0
    o.close()
    att = workloads.attempts(c["L"], R, mcs) * steps
    used = min(threads, R) if c["R"] >= threads or 2 * c["tile"] > c["L"] else threads
    desc = "%d of %d realizations, L=%d, %d MCS per step x %d step(s) + width, OpenMP threads=%d" % (
        R, c["R"], c["L"], mcs, steps, threads)
    return att / dt, used, desc, dt / steps * 1e3


def run_reference(args):
    """--impl reference: the oracle on the host cores, same metric/config; rank 0 only."""
    if int(os.environ.get("RANK", "0")) != 0:
        return
    c = workload(args)
    budget = min(150.0, max(20.0, 3.0 * args.cpu_seconds))
    v, cores, desc, ms = oracle_sample(c, budget, steps=max(1, args.steps), warmup=max(0, args.warmup))
    line = {"impl": "reference", "metric": METRIC, "value": v / 1e9, "unit": UNIT, "n_gpus": args.gpus,
            "steps": args.steps, "warmup": args.warmup, "ms_per_step": ms, "higher_is_better": True,
            "scaling": "weak", "vs_baseline": None, "dtype": "int32", "data": "synthetic",
            "config": config_dict(args, c, args.gpus),
            "cpu_baseline": {"value": v / 1e9, "unit": UNIT, "cores": cores, "kind": "oracle", "sample": desc},
            "e2e": {"value": v / 1e9, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
            "gpu_launches": 0}
    print(json.dumps(line), flush=True)


# ---------------------------------------------------------------------------------------------
# The B200 arm
# ---------------------------------------------------------------------------------------------
# Instruction roofline.  SASS count of the one-lane-per-tile attempt loop of
# thread_dt_kernel<6, 2, 1> (profiles/r2_sass_attempt_loop.md): per attempt, Philox included,
IDEAL_LOOP = {"thread_instr": 47.875, "alu_pipe": 26.125, "fma_pipe": 15.5, "lsu": 6.0, "other": 0.25}
SURVEY_FLOOR_INSTR = 22.0     # SURVEY 8(d)'s hand estimate, kept for comparison


def alu_peak_attempts_per_s(sm_count, sm_mhz):
    """Attempts/s at which the ideal loop saturates an SM sub-partition: one warp instruction issued per cycle,
    the integer alu pipe and the fma pipe each take one warp instruction per two cycles (B300_MICROARCH.md,
    'fma vs alu split', rt_SMSP = 2).  The slowest of the three binds (the alu pipe: 52.25 cycles per 32 attempts)."""
    cyc = max(IDEAL_LOOP["thread_instr"], 2.0 * IDEAL_LOOP["alu_pipe"], 2.0 * IDEAL_LOOP["fma_pipe"])
    return sm_count * 4 * 32 / cyc * sm_mhz * 1e6


def engine_peak(info, sm_mhz):
    """(peak attempts/s, where it comes from) for the update kernel of this engine, or (None, why).  The SASS count is the
    attempt loop of the lane-per-tile kernel (THREAD engine); the other engines run other loops with other limiters
    (barrier and claim rounds, vote and retry windows, bounded-draw rejection), so no instruction peak is claimed for
    them: their `frac` is null and only the engine-independent fractions (22-instruction floor, int32-equivalent sweep)
    are given."""
    if info["engine"] == "thread":
        return (alu_peak_attempts_per_s(info["sm_count"], sm_mhz),
                "derived (DESIGN.md section 6): %d SMs x 4 schedulers x 32 lanes / 52.25 cycles per 32 attempts (alu pipe of the "
                "SASS-counted loop of thread_dt_kernel<6,2,1>, profiles/r2_sass_attempt_loop.md) x %.0f MHz measured"
                % (info["sm_count"], sm_mhz))
    return None, "no SASS count for the %s engine's loop: peak not claimed" % info["engine"]


def leg_config(name):
    """name = C1..C5, 'C3/N=2', 'C5/L=256' ... -> workload dict (utils/workloads.py holds the numbers)."""
    base, _, mod = name.partition("/")
    c = dict(workloads.CONFIGS[base])
    if mod:
        k, v = mod.split("=")
        c[k] = int(v)
        if base == "C5" and k == "L":
            c["R"] = workloads.c5_realizations(c["L"])
            c["mcs"] = workloads.c5_mcs(c["L"])
    # MCS per step: 10-40 ms of device work per step, far above launch and event overheads
    dflt = {"C1": 1000, "C2": 32, "C3": 16, "C4": 4, "C5": 256, "X1": 8}[base]
    if base == "C5" and c["L"] > 64:
        dflt = {128: 256, 256: 256, 512: 128}[c["L"]]
    c["mcs_per_step"] = dflt
    return c


def run_leg(pkg, torch, name, c, steps, warmup, engine, lanes, rank, world, local, barrier, do_e2e, dist, reps=1):
    """One timed leg: `warmup` untimed steps, then `reps` timed regions of exactly `steps` steps each between CUDA events
    on the kernels' stream (barrier + synchronize on both sides, max over ranks); the region with the median time is the
    one reported.  Clocks are sampled during all timed regions."""
    import numpy as np
    L, N, R, mcs = c["L"], c["N"], c["R"], c["mcs_per_step"]
    stream = torch.cuda.Stream()
    first_real, _ = workloads.replica_range(rank, world, R)
    g = pkg.Rsos(L, N, R, c["seed"], tile=c["tile"], subsweeps=c["subsweeps"], first_real=first_real, engine=engine,
                 stream=stream.cuda_stream, lanes=lanes)
    info = g.info()
    att_step = workloads.attempts(L, R, mcs)

    def step():
        g.advance(mcs)
        return g.width()

    for _ in range(max(3, warmup)):
        step()
    barrier()
    sampler = ClockSampler(local) if rank == 0 else None
    if sampler:
        sampler.start()
        time.sleep(0.3)                                    # let nvidia-smi come up before the timed region
    g.kernel_time(True)                                    # per-advance CUDA events inside the library
    launches0 = g.info()["launches"]
    reps = max(1, reps)
    times = []
    for rep in range(reps):
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        barrier()
        if sampler and rep == 0:
            sampler.mark()
        e0.record(stream)
        for _ in range(steps):
            W2, hmean = step()
        e1.record(stream)
        barrier()
        t_rep = e0.elapsed_time(e1)
        if world > 1:
            t = torch.tensor([t_rep], dtype=torch.float64, device="cuda")
            dist.all_reduce(t, op=dist.ReduceOp.MAX)
            t_rep = float(t.item())
        times.append(t_rep)
    clocks = sampler.stop() if sampler else None
    upd_ms, upd_launches = g.kernel_time(False)            # over all `reps` regions
    launches = (g.info()["launches"] - launches0) // reps  # kernels launched inside ONE timed region of `steps` steps
    ms = sorted(times)[len(times) // 2]
    value = att_step * steps * world / (ms * 1e-3)

    # ---- e2e: host buffers through the C ABI, H2D + D2H inside the timed region -----------------
    e2e = None
    if do_e2e:
        snap = torch.empty((R, L, L), dtype=torch.int32, pin_memory=True)
        snap_np = snap.numpy()
        g.heights(out=snap_np)
        t_snap = g.t
        _, _, acc = g.sums()
        for _ in range(2):
            g.set_state(snap_np, t_snap, acc)
            step()
        barrier()
        t0 = time.perf_counter()
        for _ in range(steps):
            g.set_state(snap_np, t_snap, acc)              # H2D: R*L*L int32 + R int64
            step()                                         # advance + width (D2H: sums, accepted)
        barrier()
        dt = time.perf_counter() - t0
        if world > 1:
            t = torch.tensor([dt], dtype=torch.float64, device="cuda")
            dist.all_reduce(t, op=dist.ReduceOp.MAX)
            dt = float(t.item())
        e2e = {"value": att_step * steps * world / dt / 1e9, "unit": UNIT,
               "h2d_bytes_per_step": R * L * L * 4 + R * 8, "d2h_bytes_per_step": R * 5 * 8 + 4,
               "what": "rsos_set_state(pinned host snapshot) + rsos_advance + rsos_width per step, wall clock"}
        del snap

    # ---- roofline of the dominant kernel (the update kernel) ------------------------------------
    hbm, how = peaks()
    n_l = max(1, upd_launches)
    per_launch_att = att_step * steps * reps / n_l
    avg_ms = upd_ms / n_l
    kernel_rate = att_step * steps * reps / (upd_ms * 1e-3)   # attempts/s of the update kernels alone
    sm_mhz = (clocks or {}).get("sm_mhz") or 1965.0
    peak, peak_src = engine_peak(info, sm_mhz)
    traffic, traffic_src = traffic_note(name, info)
    sweep_gbs = kernel_rate * BYTES_PER_ATTEMPT * c["subsweeps"] / 1e9 if info["mode"] == "DT" else None
    roofline = {"bound": "alu" if peak else "latency (serial chain; no instruction count for this engine)",
                "achieved": kernel_rate / 1e9, "peak": peak / 1e9 if peak else None, "unit": "G attempts/s",
                "frac": kernel_rate / peak if peak else None, "traffic": traffic, "traffic_source": traffic_src,
                "peak_source": peak_src,
                "kernel": "update kernel, engine=%s" % info["engine"],
                "attempts_per_launch": per_launch_att, "avg_launch_ms": avg_ms, "update_launches": int(upd_launches),
                "update_share_of_step": upd_ms / sum(times),
                "frac_of_survey_floor_22_instr": kernel_rate / (info["sm_count"] * 4 * 32 * sm_mhz * 1e6 / SURVEY_FLOOR_INSTR),
                # north_star's other candidate, kept as a labelled int32-EQUIVALENT sweep rate: the packed working
                # lattice moves far fewer bytes (see traffic), so this is not what binds
                "int32_equiv_sweep": {"bytes_per_attempt": BYTES_PER_ATTEMPT * c["subsweeps"], "GBps": sweep_gbs,
                                      "hbm_peak_GBps": hbm, "peak_source": how,
                                      "frac": (sweep_gbs / hbm) if sweep_gbs else None}}
    out = {"workload": name, "value": value / 1e9, "unit": UNIT, "steps": steps, "warmup": max(3, warmup), "reps": reps,
           "region_ms": times, "ms_per_step": ms / steps, "config": config_dict_for(name, c, world), "residency": l2_note(c, info),
           "engine": info, "clocks": clocks, "e2e": e2e,
           "gpu_launches": int(launches), "roofline": roofline,
           "result_check": {"W2_mean": float(np.mean(W2)), "hmean_mean": float(np.mean(hmean)), "t_mcs": int(g.t)}}
    g.close()
    return out


def run_seeds4(pkg, torch, c, steps, warmup, reps):
    """BASELINE.json configs[1] as it is worded ("seeds 1..4"): the four 128-realization runs advance together, one
    context per seed, each on its own stream, so that a colour pass has four times the tiles in flight.  A step = every
    context's rsos_advance(mcs_per_step), then every context's rsos_width.  Device-timed from an event recorded while
    all streams are idle to one recorded after the last width has synchronised its stream.  One GPU only."""
    L, N, R, mcs = c["L"], c["N"], c["R"], c["mcs_per_step"]
    seeds = (1, 2, 3, 4)
    streams = [torch.cuda.Stream() for _ in seeds]
    ctxs = [pkg.Rsos(L, N, R, sd, tile=c["tile"], subsweeps=c["subsweeps"], stream=st.cuda_stream) for sd, st in zip(seeds, streams)]

    def step():
        for g in ctxs:
            g.advance(mcs)
        return [g.width() for g in ctxs]

    for _ in range(max(3, warmup)):
        step()
    times = []
    for _ in range(max(1, reps)):
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        torch.cuda.synchronize()
        e0.record(streams[0])
        for _ in range(steps):
            step()
        e1.record(streams[0])
        torch.cuda.synchronize()
        times.append(e0.elapsed_time(e1))
    ms = sorted(times)[len(times) // 2]
    launches = sum(g.info()["launches"] for g in ctxs)
    for g in ctxs:
        g.close()
    att = workloads.attempts(L, R, mcs) * len(seeds) * steps
    return {"workload": "C2 seeds 1..4", "value": att / (ms * 1e-3) / 1e9, "unit": UNIT, "steps": steps, "reps": reps,
            "region_ms": times, "ms_per_step": ms / steps, "contexts": len(seeds), "launches_total": int(launches),
            "what": "4 contexts (seeds 1..4) on 4 streams, advance all then width all"}


def oracle_side_timings():
    """The two other oracle timings SURVEY 8(d) / BASELINE.md section 3 list (G attempts/s each): a cut-down C4 (L = 32768,
    one surface, 2 MCS) on all cores, and C1 in full on one thread.  The all-cores run comes first and names its thread
    count: the oracle's thread setting is process-wide, so a one-thread run would otherwise carry over."""
    from oracle import rsos_oracle
    rsos_oracle.build()
    out = {}
    cores = os.cpu_count() or 1
    c4 = workloads.CONFIGS["C4"]
    try:
        o = rsos_oracle.Oracle(c4["L"], c4["N"], 1, c4["seed"], tile=c4["tile"], subsweeps=c4["subsweeps"], threads=cores)
        t0 = time.perf_counter()
        o.advance(2)
        o.width()
        out["c4_cut_2mcs_allcores"] = workloads.attempts(c4["L"], 1, 2) / (time.perf_counter() - t0) / 1e9
        o.close()
    except (MemoryError, RuntimeError, ValueError) as e:   # 4 GiB of heights did not fit on this host
        out["c4_cut_2mcs_allcores"] = None
        out["c4_cut_error"] = str(e)[:80]
    c1 = workloads.CONFIGS["C1"]
    o = rsos_oracle.Oracle(c1["L"], c1["N"], c1["R"], c1["seed"], tile=c1["tile"], subsweeps=c1["subsweeps"], threads=1)
    t0 = time.perf_counter()
    o.advance(c1["mcs"])
    o.width()
    out["c1_full_1thread"] = workloads.attempts(c1["L"], c1["R"], c1["mcs"]) / (time.perf_counter() - t0) / 1e9
    o.close()
    return out


def r6(x):
    """Six significant digits: keeps the final line short."""
    return float("%.6g" % x) if isinstance(x, float) else x


def make_line(c, world, steps, warmup, head, cpu=None, c4=None, seeds4=None, legs_file=None):
    """The ONE final stdout line: the headline leg `head` (a run_leg record) reduced to the keys the contract names,
    plus compact side numbers.  Must stay below MAX_LINE_BYTES; optional parts are dropped, last first, if it does not."""
    rf, ie = head["roofline"], head["roofline"]["int32_equiv_sweep"]
    ck = head["clocks"] or {}
    line = {"metric": METRIC, "value": r6(head["value"]), "unit": UNIT, "n_gpus": world, "steps": steps,
            "warmup": max(3, warmup), "ms_per_step": r6(head["ms_per_step"]), "higher_is_better": True, "scaling": "weak",
            "vs_baseline": None, "dtype": "int32", "data": "synthetic", "config": head["config"], "reps": head["reps"],
            "clocks": {k: ck.get(k) for k in ("sm_mhz", "sm_max_mhz", "reasons", "samples")},
            "e2e": None if not head["e2e"] else {k: r6(head["e2e"][k]) for k in ("value", "unit", "h2d_bytes_per_step", "d2h_bytes_per_step")},
            "gpu_launches": head["gpu_launches"],
            "roofline": {"bound": rf["bound"], "achieved": r6(rf["achieved"]), "peak": r6(rf["peak"]), "unit": rf["unit"],
                         "frac": r6(rf["frac"]), "traffic": rf["traffic"],
                         "kernel": "%s engine, %d lanes/tile, %d bits/site" % (head["engine"]["engine"], head["engine"].get("lanes", 0),
                                                                              head["engine"].get("packed_bits", 0)),
                         "avg_launch_ms": r6(rf["avg_launch_ms"]), "attempts_per_launch": int(rf["attempts_per_launch"]),
                         "update_share_of_step": r6(rf["update_share_of_step"]),
                         "frac_hbm_int32_equiv": r6(ie["frac"]),
                         "frac_of_survey_floor_22_instr": r6(rf["frac_of_survey_floor_22_instr"]),
                         "peak_source": "DESIGN.md 6"},
            "cpu_baseline": None if not cpu else {k: r6(v) for k, v in cpu.items()}}
    if c4:
        line["c4"] = {"value": r6(c4["value"]), "kernel": r6(c4["roofline"]["achieved"]), "frac": r6(c4["roofline"]["frac"]),
                      "frac_hbm_int32_equiv": r6(c4["roofline"]["int32_equiv_sweep"]["frac"]),
                      "e2e": r6(c4["e2e"]["value"]) if c4.get("e2e") else None}
    if seeds4:
        line["c2_seeds4"] = {"value": r6(seeds4["value"]), "ms_per_step": r6(seeds4["ms_per_step"]), "what": "4 contexts, 4 streams"}
    if legs_file:
        line["legs_file"] = os.path.basename(legs_file)
    for drop in ("legs_file", "c2_seeds4", "c4"):
        if len(json.dumps(line)) < MAX_LINE_BYTES:
            break
        line.pop(drop, None)
    if len(json.dumps(line)) >= MAX_LINE_BYTES:
        raise RuntimeError("bench.py: final line is %d bytes (limit %d)" % (len(json.dumps(line)), MAX_LINE_BYTES))
    return line


def run_b200(args):
    import torch
    import torch.distributed as dist
    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device; the hot path has no CPU fallback")
    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    torch.cuda.set_device(local)
    if world > 1:
        dist.init_process_group("nccl", device_id=torch.device("cuda", local))

    def barrier():
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    from paper_1605_02620_b200 import build as _build
    if rank == 0:
        _build.build()
    barrier()
    import paper_1605_02620_b200 as pkg

    c = workload(args)
    engine = {"auto": 0, "simple": 1, "warp": 2, "onchip": 3, "thread": 4, "resident": 5, "fine": 6, "level": 8}[args.engine]
    head = run_leg(pkg, torch, args.workload, c, args.steps, args.warmup, engine, args.lanes, rank, world, local, barrier,
                   not args.no_e2e, dist, reps=args.reps)

    # ---- side legs (one GPU only): full records go to the side file, two compact numbers to the final line ----------
    legs, seeds4 = {}, None
    if world == 1 and not args.no_extra:
        for name in (EXTRA_LEGS if args.all_legs else DEFAULT_LEGS):
            if name == args.workload:
                continue
            legs[name] = run_leg(pkg, torch, name, leg_config(name), args.extra_steps, 3, 0, 0, rank, world, local, barrier,
                                 not args.no_e2e, dist, reps=args.reps)
        if args.workload == "C2":
            seeds4 = run_seeds4(pkg, torch, c, max(1, args.steps // 2), 3, args.reps)

    if rank != 0:
        if world > 1:
            dist.destroy_process_group()
        return

    cpu = None
    if not args.no_cpu_baseline and world == 1:
        v, cores, desc, _ = oracle_sample(c, args.cpu_seconds)
        cpu = {"value": v / 1e9, "unit": UNIT, "cores": cores, "kind": "oracle", "sample": desc}
        cpu.update(oracle_side_timings())

    try:
        with open(args.legs_file, "w") as f:
            json.dump({"headline": head, "legs": legs, "c2_seeds4": seeds4, "cpu_baseline": cpu, "cpu_model": cpu_model()}, f, indent=1)
        legs_file = args.legs_file
    except OSError:
        legs_file = None
    line = make_line(c, world, args.steps, args.warmup, head, cpu, legs.get("C4"), seeds4, legs_file)
    print(json.dumps(line), flush=True)
    if world > 1:
        dist.destroy_process_group()


def main():
    args = parse()
    if args.impl == "reference":
        run_reference(args)
    else:
        run_b200(args)


if __name__ == "__main__":
    main()
