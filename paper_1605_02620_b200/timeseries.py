"""W^2(t) time series of a named workload through the C ABI (north_star: "W^2 ... taken at log-spaced times";
SURVEY section 5: per-measurement rows; Eq. 10).

    python -m paper_1605_02620_b200.timeseries C2 [--out c2.jsonl] [--schedule log64|eq10|every] [--tmax T]
                                                  [--moments] [--R r] [--seed s] [--seeds 1,2,3,4]

One JSONL row per measurement time and realization: {"t", "r", "S1", "S2", "accepted"} (exact integers, Eq. 2 follows
from them: W2 = (L^2 S2 - S1^2) / L^4), with "phi2", "phi3", "phi4" (Eq. 13) added by --moments; a header row names
the run.  The last line printed is a summary: <W^2>(t) with its standard error and the effective exponent beta_eff
(Eq. 9).  Everything is computed by the library's kernels; this module only calls rsos_advance / rsos_sums /
rsos_height_moments at the listed times and writes what they return.
"""
import argparse
import json
import sys

import numpy as np

from . import analysis
from .utils import workloads


def measurement_times(schedule, t_max):
    if schedule == "log64":
        return workloads.log_spaced_times(t_max)
    if schedule == "eq10":
        return workloads.eq10_times(t_max)
    if schedule == "every":
        return list(range(1, int(t_max) + 1))
    raise ValueError("unknown schedule %r" % schedule)


def run(pkg, cfg, times, out=None, moments=False, engine=0):
    """Advance a fresh context of workload dict `cfg` (L, N, R, seed, tile, subsweeps) to each of the ascending
    `times`, taking the exact sums there.  Returns (times, W2[len(times), R], hmean[len(times), R]); writes JSONL rows
    to the open text file `out` if given."""
    g = pkg.Rsos(cfg["L"], cfg["N"], cfg["R"], cfg["seed"], tile=cfg["tile"], subsweeps=cfg["subsweeps"],
                 first_real=cfg.get("first_real", 0), engine=engine)
    if out is not None:
        out.write(json.dumps({"header": True, "config": {k: cfg[k] for k in ("L", "N", "R", "seed", "tile", "subsweeps")},
                              "engine": g.info()["engine"], "schedule_mode": g.info()["mode"]}) + "\n")
    W2s, hms, t = [], [], 0
    for tm in times:
        tm = int(tm)
        if tm < t:
            raise ValueError("measurement times must ascend")
        g.advance(tm - t)
        t = tm
        S1, S2, acc = g.sums()
        W2, hm = g.width()
        W2s.append(W2)
        hms.append(hm)
        if out is not None:
            phi = g.height_moments()[1] if moments else None
            for r in range(cfg["R"]):
                row = {"t": t, "r": cfg.get("first_real", 0) + r, "S1": int(S1[r]), "S2": int(S2[r]), "accepted": int(acc[r])}
                if phi is not None:
                    row.update(phi2=float(phi[r, 0]), phi3=float(phi[r, 1]), phi4=float(phi[r, 2]))
                out.write(json.dumps(row) + "\n")
    g.close()
    return list(times), np.array(W2s), np.array(hms)


def run_seeds(pkg, cfg, seeds, times, out=None):
    """BASELINE.json configs[1] asks for "seeds 1..4": the same workload once per seed.  This runs them TOGETHER -- one
    context per seed, each on its own CUDA stream; rsos_advance only enqueues, so all contexts' kernels are in flight at once
    -- which is how a config with few tiles per colour pass fills the GPU (C2: 304 against 197 G attempts/s on a B200,
    DESIGN.md section 11).  Each seed's run is the same pure function of (seed, r, ...) as a lone run; only the wall time
    changes.  Returns (times, W2[len(seeds), len(times), R]); JSONL rows carry a "seed" field."""
    import torch
    streams = [torch.cuda.Stream() for _ in seeds]
    ctxs = [pkg.Rsos(cfg["L"], cfg["N"], cfg["R"], sd, tile=cfg["tile"], subsweeps=cfg["subsweeps"],
                     first_real=cfg.get("first_real", 0), stream=st.cuda_stream) for sd, st in zip(seeds, streams)]
    if out is not None:
        out.write(json.dumps({"header": True, "config": {k: cfg[k] for k in ("L", "N", "R", "tile", "subsweeps")},
                              "seeds": list(seeds), "engine": ctxs[0].info()["engine"]}) + "\n")
    W2s, t = [[] for _ in seeds], 0
    for tm in times:
        tm = int(tm)
        if tm < t:
            raise ValueError("measurement times must ascend")
        for g in ctxs:
            g.advance(tm - t)                              # asynchronous: enqueued on every stream before any read-back
        t = tm
        for i, (sd, g) in enumerate(zip(seeds, ctxs)):
            S1, S2, acc = g.sums()
            W2s[i].append(g.width()[0])
            if out is not None:
                for r in range(cfg["R"]):
                    out.write(json.dumps({"t": t, "seed": int(sd), "r": cfg.get("first_real", 0) + r, "S1": int(S1[r]),
                                          "S2": int(S2[r]), "accepted": int(acc[r])}) + "\n")
    for g in ctxs:
        g.close()
    return list(times), np.array(W2s)


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("workload", help="C1..C5 (paper_1605_02620_b200/utils/workloads.py)")
    ap.add_argument("--out", default="")
    ap.add_argument("--schedule", default="", choices=["", "log64", "eq10", "every"])
    ap.add_argument("--tmax", type=int, default=0)
    ap.add_argument("--R", type=int, default=0)
    ap.add_argument("--seed", type=int, default=0)
    ap.add_argument("--moments", action="store_true")
    ap.add_argument("--seeds", default="", help="e.g. 1,2,3,4: run these seeds together, one context and stream each")
    a = ap.parse_args()
    import paper_1605_02620_b200 as pkg
    cfg = dict(workloads.CONFIGS[a.workload])
    if a.R:
        cfg["R"] = a.R
    if a.seed:
        cfg["seed"] = a.seed
    t_max = a.tmax or cfg["mcs"]
    schedule = a.schedule or ("every" if a.workload == "C1" else "log64")
    times = measurement_times(schedule, t_max)
    f = open(a.out, "w") if a.out else None
    if a.seeds:
        seeds = [int(x) for x in a.seeds.split(",")]
        try:
            ts, W2 = run_seeds(pkg, cfg, seeds, times, out=f)
        finally:
            if f:
                f.close()
        w2m = W2.mean(axis=(0, 2))                           # over seeds and realizations
        bt, be = analysis.beta_eff(ts, w2m)
        json.dump({"workload": a.workload, "schedule": schedule, "seeds": seeds, "times": ts, "W2_mean": w2m.tolist(),
                   "W2_stderr": [analysis.standard_error(W2[:, i, :].ravel()) for i in range(len(ts))],
                   "beta_eff": {"t": bt.tolist(), "beta": be.tolist()}}, sys.stdout)
        sys.stdout.write("\n")
        return
    try:
        ts, W2, hm = run(pkg, cfg, times, out=f, moments=a.moments)
    finally:
        if f:
            f.close()
    w2m = W2.mean(axis=1)
    bt, be = analysis.beta_eff(ts, w2m)
    summary = {"workload": a.workload, "schedule": schedule, "times": ts, "W2_mean": w2m.tolist(),
               "W2_stderr": [analysis.standard_error(w) for w in W2], "hmean_mean": hm.mean(axis=1).tolist(),
               "beta_eff": {"t": bt.tolist(), "beta": be.tolist()}}
    json.dump(summary, sys.stdout)
    sys.stdout.write("\n")


if __name__ == "__main__":
    main()
