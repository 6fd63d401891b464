"""Domain-decomposition consistency table (the analogue of the paper's Fig. 5 / P:202-208):
ensemble <W^2>(t) and <h>(t) of the seeded schedule DT(S, K) for several tile sides S against serial
random-sequential deposition (RS mode: one tile = the lattice) at the same L, N and number of realizations.

    python -m paper_1605_02620_b200.dd_consistency [--L 128] [--N 1] [--R 4096] [--times 1 10 100] [--seed 1]

Runs entirely through the C ABI on the GPU (no oracle).  One row per schedule; deviations are relative to
RS, with the standard error of the mean of both ensembles combined (reading Q9).  The smallest
sequential unit sets the bias (Q8); S = 64 is what the hot path uses.  K = "P" is the
Poisson variant DTP(c).  The last column is the update throughput of the schedule on
this ensemble (CUDA events inside the library, rsos_kernel_time).
"""
import argparse
import math

import numpy as np


def ensemble(pkg, L, N, R, seed, tile, K, times):
    """([(mean W2, SE, mean h, SE)] at the given times (MCS), info, G attempts/s of the update kernels) for one
    schedule; K = "P": the Poisson variant."""
    kw = dict(tile=tile, poisson=True) if K == "P" else dict(tile=tile, subsweeps=K)
    g = pkg.Rsos(L, N, R, seed, **kw)
    g.kernel_time(True)
    out, t = [], 0
    for tt in times:
        g.advance(tt - t)
        t = tt
        w2, hm = g.width()
        out.append((w2.mean(), w2.std(ddof=1) / math.sqrt(R), hm.mean(), hm.std(ddof=1) / math.sqrt(R)))
    ms, _ = g.kernel_time(False)
    info = g.info()
    g.close()
    return out, info, float(L) * L * R * t / (ms * 1e-3) / 1e9


def table(L=128, N=1, R=4096, seed=1, times=(1, 10, 100),
          schedules=((8, 1), (16, 1), (32, 1), (64, 1), (32, 4), (64, 4), (8, "P"), (16, "P"))):
    import paper_1605_02620_b200 as pkg
    ref, info, rate = ensemble(pkg, L, N, R, seed, L, 1, times)       # 2S > L: serial RS
    assert info["mode"] == "RS"
    rows = [("RS (serial)", info["engine"], ref, None, rate)]
    for S, K in schedules:
        if 2 * S > L:
            continue
        res, info, rate = ensemble(pkg, L, N, R, seed + 1000 * S + (77 if K == "P" else K), S, K, times)   # independent ensemble
        dev = []
        for (w, sw, h, sh), (w0, sw0, h0, sh0) in zip(res, ref):
            dev.append(((w - w0) / w0, math.hypot(sw, sw0) / w0, (h - h0) / h0, math.hypot(sh, sh0) / h0))
        rows.append(("DTP(%d)" % S if K == "P" else "DT(%d,%d)" % (S, K), info["engine"], res, dev, rate))
    return rows


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--L", type=int, default=128)
    ap.add_argument("--N", type=int, default=1)
    ap.add_argument("--R", type=int, default=4096)
    ap.add_argument("--seed", type=int, default=1)
    ap.add_argument("--times", type=int, nargs="+", default=[1, 10, 100])
    a = ap.parse_args()
    rows = table(a.L, a.N, a.R, a.seed, tuple(a.times))
    print("L = %d, N = %d, %d realizations per schedule; W2 (relative deviation from RS, in units of the combined SE)" % (a.L, a.N, a.R))
    print("| schedule | engine | " + " | ".join("t = %d" % t for t in a.times) + " | G attempts/s |")
    print("|---|---|" + "---|" * (len(a.times) + 1))
    for name, eng, res, dev, rate in rows:
        cells = []
        for i, (w, sw, h, sh) in enumerate(res):
            if dev is None:
                cells.append("%.6f(%.0f) / h %.5f" % (w, sw * 1e6, h))
            else:
                dw, sdw, dh, sdh = dev[i]
                cells.append("%.6f (%+.2f %%, %.1f SE) / h %+.3f %%" % (w, 100 * dw, abs(dw) / sdw, 100 * dh))
        print("| %s | %s | " % (name, eng) + " | ".join(cells) + " | %.0f |" % rate)


if __name__ == "__main__":
    main()
