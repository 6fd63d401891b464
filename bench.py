#!/usr/bin/env python
"""bench.py -- RSOS site-update attempts per second on B200 (BASELINE.json metric), one JSON line.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--workload C2|C4|C3/N=2|C5/L=256|...] [--impl reference]

A *step* is one pass of the whole hot path over one
batch: `mcs_per_step` Monte-Carlo steps of rsos_advance (Philox draws, origin draw, tile staging,
attempt loop, write-back) followed by one rsos_width (int64 width reduction, result read to host).
The headline workload is BASELINE.json configs[1] (C2: L=1024, N=1, 128 realizations, DT(64,1)).  The
same run then times, with the same fields under "extra", the other north_star config (C4: L=2^15, one
surface), short legs on C3 (N=1, 2), C5 (L=64..512) and C1, and one on the paper's own largest lattice
(X1: L=9605, not a power of two), so that every BASELINE config has a
number the driver's own run produced.  Nothing is flushed between steps: a step sweeps the same
resident lattice 4K * mcs_per_step times exactly as a production run does; `config.l2` says what is
resident where.

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
cpu_baseline / --impl reference: the CPU oracle as it stands, on a bounded sample of the workload.
N > 1: replicas only: rank i runs realizations [i*R, (i+1)*R), no collective
on the data path; scaling is weak; the extra legs are skipped.
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
    ap.add_argument("--no-extra", action="store_true", help="skip the legs on the other BASELINE configs")
    ap.add_argument("--extra-steps", type=int, default=5, help="timed steps of each extra leg")
    ap.add_argument("--cpu-seconds", type=float, default=12.0, help="target CPU time of the oracle sample")
    return ap.parse_args()


# legs of the default run besides the headline workload: the other north_star config (C4) and short legs on the rest
EXTRA_LEGS = ("C4", "C2", "C3", "C3/N=2", "C5", "C5/L=128", "C5/L=256", "C5/L=512", "C1", "X1")


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
    """Timing rule: say whether the inputs exceed L2 or are flushed.  A step sweeps the same resident lattice
    mcs_per_step * 4K times, exactly as a production run does, so nothing is flushed; what is resident is stated."""
    int32_mib = c["R"] * c["L"] ** 2 * 4 / 2 ** 20
    if info and info.get("engine") == "resident":
        return ("lattice resident in shared memory for all %d MCS of a step (packed copy in HBM %.0f MiB, touched once per "
                "rsos_advance); nothing to flush" % (c["mcs_per_step"], int32_mib * info.get("packed_bits", 2) / 32))
    if info and info.get("engine") == "thread":
        fb = 2 if (c["N"] <= 1 and c["tile"] >= 16) else 4
        work = int32_mib * fb / 32
        return ("working lattice %.0f MiB per GPU (%d bits/site, DESIGN.md section 5; int32 view %.0f MiB) vs 126 MB L2: %s; "
                "no flush: consecutive sweeps of a production run see the same residency" % (
                    work, fb, int32_mib, "larger than L2" if work * 2 ** 20 > 126e6 else "L2-resident by design"))
    return "state %.0f MiB int32 per GPU vs 126 MB L2: %s" % (
        int32_mib, "inputs larger than L2, no flush" if int32_mib * 2 ** 20 > 2 * 126e6 else "L2/on-chip resident by design")


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
    return {"workload": "%s: RSOS N=%d, L=%d periodic, %d realizations per GPU, int32 heights, flat start, seed %d"
                        % (name, c["N"], c["L"], c["R"], c["seed"]),
            "schedule": mode, "mcs_per_step": c["mcs_per_step"],
            "step": "rsos_advance(mcs_per_step) + rsos_width",
            "l2": l2_note(c, info),
            "parallelism": "replicas x%d (independent realizations, no collective)" % n_gpus}


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
            "cpu_baseline": {"value": v / 1e9, "unit": UNIT, "cores": cores, "cpu_model": cpu_model(), "kind": "oracle",
                             "sample": desc},
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


def run_leg(pkg, torch, name, c, steps, warmup, engine, lanes, rank, world, local, barrier, do_e2e, dist):
    """One timed leg: `warmup` untimed steps, then exactly `steps` steps between CUDA events on the kernels' stream
    (barrier + synchronize on both sides, max over ranks), clocks sampled during the timed region."""
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
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    barrier()
    if sampler:
        sampler.mark()
    e0.record(stream)
    for _ in range(steps):
        W2, hmean = step()
    e1.record(stream)
    barrier()
    ms = e0.elapsed_time(e1)
    clocks = sampler.stop() if sampler else None
    upd_ms, upd_launches = g.kernel_time(False)
    launches = g.info()["launches"] - launches0
    if world > 1:
        t = torch.tensor([ms], dtype=torch.float64, device="cuda")
        dist.all_reduce(t, op=dist.ReduceOp.MAX)
        ms = float(t.item())
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
    per_launch_att = att_step * steps / n_l
    avg_ms = upd_ms / n_l
    kernel_rate = att_step * steps / (upd_ms * 1e-3)       # attempts/s of the update kernels alone
    sm_mhz = (clocks or {}).get("sm_mhz") or 1965.0
    peak = alu_peak_attempts_per_s(info["sm_count"], sm_mhz)
    traffic, traffic_src = traffic_note(name, info)
    sweep_gbs = kernel_rate * BYTES_PER_ATTEMPT * c["subsweeps"] / 1e9 if info["mode"] == "DT" else None
    roofline = {"bound": "alu", "achieved": kernel_rate / 1e9, "peak": peak / 1e9, "unit": "G attempts/s",
                "frac": kernel_rate / peak, "traffic": traffic, "traffic_source": traffic_src,
                "peak_source": "derived (DESIGN.md section 6): %d SMs x 4 schedulers x 32 lanes / 52.25 cycles per 32 attempts "
                               "(alu pipe of the SASS-counted ideal loop, profiles/r2_sass_attempt_loop.md) x %.0f MHz measured"
                               % (info["sm_count"], sm_mhz),
                "kernel": "update kernel, engine=%s" % info["engine"],
                "attempts_per_launch": per_launch_att, "avg_launch_ms": avg_ms, "update_launches": int(upd_launches),
                "update_share_of_step": upd_ms / ms,
                "frac_of_survey_floor_22_instr": kernel_rate / (info["sm_count"] * 4 * 32 * sm_mhz * 1e6 / SURVEY_FLOOR_INSTR),
                # north_star's other candidate, kept as a labelled int32-EQUIVALENT sweep rate: the packed working
                # lattice moves far fewer bytes (see traffic), so this is not what binds
                "int32_equiv_sweep": {"bytes_per_attempt": BYTES_PER_ATTEMPT * c["subsweeps"], "GBps": sweep_gbs,
                                      "hbm_peak_GBps": hbm, "peak_source": how,
                                      "frac": (sweep_gbs / hbm) if sweep_gbs else None}}
    out = {"workload": name, "value": value / 1e9, "unit": UNIT, "steps": steps, "warmup": max(3, warmup),
           "ms_per_step": ms / steps, "config": None, "engine": info, "clocks": clocks, "e2e": e2e,
           "gpu_launches": int(launches), "roofline": roofline,
           "result_check": {"W2_mean": float(np.mean(W2)), "hmean_mean": float(np.mean(hmean)), "t_mcs": int(g.t)}}
    g.close()
    return out


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
                   not args.no_e2e, dist)

    # ---- the other BASELINE configs, same fields, fewer steps (one GPU only) -------------------------
    extra = {}
    if world == 1 and not args.no_extra:
        for name in EXTRA_LEGS:
            if name == args.workload:
                continue
            ce = leg_config(name)
            leg = run_leg(pkg, torch, name, ce, args.extra_steps, 3, 0, 0, rank, world, local, barrier,
                          not args.no_e2e, dist)
            leg["config"] = config_dict_for(name, ce, 1, leg["engine"])
            extra[name] = leg

    if rank != 0:
        if world > 1:
            dist.destroy_process_group()
        return

    cpu = None
    if not args.no_cpu_baseline and world == 1:
        v, cores, desc, _ = oracle_sample(c, args.cpu_seconds)
        cpu = {"value": v / 1e9, "unit": UNIT, "cores": cores, "cpu_model": cpu_model(), "kind": "oracle", "sample": desc}

    line = {"metric": METRIC, "value": head["value"], "unit": UNIT, "n_gpus": world, "steps": args.steps,
            "warmup": max(3, args.warmup), "ms_per_step": head["ms_per_step"], "higher_is_better": True, "scaling": "weak",
            "vs_baseline": None, "dtype": "int32", "data": "synthetic", "config": config_dict(args, c, world, head["engine"]),
            "engine": head["engine"], "clocks": head["clocks"], "e2e": head["e2e"], "gpu_launches": head["gpu_launches"],
            "roofline": head["roofline"], "cpu_baseline": cpu, "result_check": head["result_check"], "extra": extra}
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
