"""Stationary-regime roughness (BASELINE.json configs[4], the paper's Sec. III.B): for L in
64..512 run R = 2^24 / L^2 realizations to t = 20 L^1.6 MCS and average W^2 over the last 25 % of the run;
the slope of ln W_sat vs ln L estimates the roughness exponent alpha (paper: 0.390(4)).

    python -m paper_1605_02620_b200.saturation [--N 1] [--sizes 64 128 256 512] [--samples 100]

Runs entirely through the C ABI on the GPU (L = 64: serial RS on chip; L >= 128: DT(64,4)).
"""
import argparse
import math
import time

import numpy as np

from .utils import workloads


def w2_sat(pkg, L, N, seed=1, samples=100, tile=64, subsweeps=4):
    R = workloads.c5_realizations(L)
    tmax = workloads.c5_mcs(L)
    g = pkg.Rsos(L, N, R, seed, tile=tile, subsweeps=subsweeps)
    info = g.info()
    t0 = tmax - tmax // 4
    g.advance(t0)
    step = max(1, (tmax - t0) // samples)
    acc, n, t = 0.0, 0, t0
    while t + step <= tmax:
        g.advance(step)
        t += step
        acc += float(g.width()[0].mean())
        n += 1
    g.close()
    return acc / n, R, tmax, info


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--N", type=int, default=1)
    ap.add_argument("--sizes", type=int, nargs="+", default=[64, 128, 256, 512])
    ap.add_argument("--samples", type=int, default=100)
    a = ap.parse_args()
    import paper_1605_02620_b200 as pkg
    rows = []
    for L in a.sizes:
        t0 = time.perf_counter()
        w2, R, tmax, info = w2_sat(pkg, L, a.N, samples=a.samples)
        dt = time.perf_counter() - t0
        rows.append((L, w2))
        print("L = %4d  R = %5d  t = %7d MCS  %s/%s  <W2>_sat = %.5f  W_sat = %.5f  (%.1f s, %.1f G attempts/s)" % (
            L, R, tmax, info["mode"], info["engine"], w2, math.sqrt(w2), dt, workloads.attempts(L, R, tmax) / dt / 1e9), flush=True)
    if len(rows) >= 2:
        x = np.log([r[0] for r in rows])
        y = 0.5 * np.log([r[1] for r in rows])
        print("alpha (slope of ln W_sat vs ln L) = %.4f; successive pairs: %s" % (
            np.polyfit(x, y, 1)[0], ", ".join("%.4f" % s for s in np.diff(y) / np.diff(x))))


if __name__ == "__main__":
    main()
