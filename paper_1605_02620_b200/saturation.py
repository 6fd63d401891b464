"""Stationary-regime roughness (BASELINE.json configs[4], the paper's Sec. III.B): for L in
64..512 run R = 2^24 / L^2 realizations to t = 20 L^1.6 MCS and average W^2 over the last 25 % of the run;
the slope of ln W_sat vs ln L estimates the roughness exponent alpha (paper: 0.390(4)), Eq. (8) gives the
effective exponents.  With --moments the same samples give the shape measures of the steady state (S 8(f) NEXT-2,
Eq. 13-15): skewness / kurtosis of the width distribution P(W^2) over realizations and times (paper:
S = 1.70(1), Q = 5.38(4)) and of the height distribution (S_h = 0.270(5), Q_h = 0.15(1)).

    python -m paper_1605_02620_b200.saturation [--N 1] [--sizes 64 128 256 512] [--samples 100] [--moments]

Runs entirely through the C ABI on the GPU (L = 64: serial RS on chip; L >= 128: DT(64,4)).
"""
import argparse
import math
import time

import numpy as np

from . import analysis
from .utils import workloads


def steady_state(pkg, L, N, seed=1, samples=100, tile=64, subsweeps=4, R=None, tmax=None, moments=False):
    """Run to tmax (default 20 L^1.6) and sample the last 25 % of the run `samples` times.  Returns a dict:
    W2 [samples, R], phi [samples, R, 3] (Eq. 13 per surface; only with moments), R, tmax, info."""
    R = R or workloads.c5_realizations(L)
    tmax = tmax or workloads.c5_mcs(L)
    g = pkg.Rsos(L, N, R, seed, tile=tile, subsweeps=subsweeps)
    info = g.info()
    t0 = tmax - tmax // 4
    g.advance(t0)
    step = max(1, (tmax - t0) // samples)
    W2s, phis, t = [], [], t0
    while t + step <= tmax:
        g.advance(step)
        t += step
        W2s.append(g.width()[0])
        if moments:
            phis.append(g.height_moments()[1])
    g.close()
    return {"W2": np.array(W2s), "phi": np.array(phis) if moments else None, "R": R, "tmax": tmax, "info": info}


def shape_measures(res):
    """(S, Q) of P(W^2) and (S_h, Q_h) of the height distribution from a steady_state(..., moments=True) result."""
    S, Q = analysis.distribution_shape(res["W2"])
    S_h, Q_h = analysis.height_distribution_shape(res["phi"])
    return {"S": S, "Q": Q, "S_h": S_h, "Q_h": Q_h}


def w2_sat(pkg, L, N, seed=1, samples=100, tile=64, subsweeps=4):
    res = steady_state(pkg, L, N, seed=seed, samples=samples, tile=tile, subsweeps=subsweeps)
    return float(res["W2"].mean()), res["R"], res["tmax"], res["info"]


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--N", type=int, default=1)
    ap.add_argument("--sizes", type=int, nargs="+", default=[64, 128, 256, 512])
    ap.add_argument("--samples", type=int, default=100)
    ap.add_argument("--moments", action="store_true", help="also S, Q of P(W^2) and S_h, Q_h of the heights (Eq. 13-15)")
    a = ap.parse_args()
    import paper_1605_02620_b200 as pkg
    rows = []
    for L in a.sizes:
        t0 = time.perf_counter()
        res = steady_state(pkg, L, a.N, samples=a.samples, moments=a.moments)
        w2, R, tmax, info = float(res["W2"].mean()), res["R"], res["tmax"], res["info"]
        dt = time.perf_counter() - t0
        rows.append((L, w2))
        print("L = %4d  R = %5d  t = %7d MCS  %s/%s  <W2>_sat = %.5f  W_sat = %.5f  (%.1f s, %.1f G attempts/s)" % (
            L, R, tmax, info["mode"], info["engine"], w2, math.sqrt(w2), dt, workloads.attempts(L, R, tmax) / dt / 1e9), flush=True)
        if a.moments:
            m = shape_measures(res)
            print("          width distribution S = %.3f, Q = %.3f (paper 1.70(1), 5.38(4));  heights S_h = %.4f, Q_h = %.4f "
                  "(paper 0.270(5), 0.15(1))" % (m["S"], m["Q"], m["S_h"], m["Q_h"]), flush=True)
    if len(rows) >= 2:
        x = np.log([r[0] for r in rows])
        y = 0.5 * np.log([r[1] for r in rows])
        _, ae = analysis.alpha_eff([r[0] for r in rows], [r[1] for r in rows])
        print("alpha (slope of ln W_sat vs ln L) = %.4f; alpha_eff (Eq. 8) of successive sizes: %s" % (
            np.polyfit(x, y, 1)[0], ", ".join("%.4f" % s for s in ae)))


if __name__ == "__main__":
    main()
