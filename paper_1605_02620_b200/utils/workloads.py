"""Seeded synthetic workloads (BASELINE.json configs C1..C5) and measurement-time schedules.

Shared by tests, bench.py and the oracle harness.  Holds NONE of the method's arithmetic: an RSOS
workload is fully described by (L, N, R, seed, tile S, sub-sweeps K, MCS); the lattice starts flat
 and every random number is drawn inside the implementations from Philox.
"""
import math

# name -> dict(L, N, R, mcs, seed, tile, subsweeps); lists mean "one run per entry"
CONFIGS = {
    "C1": dict(L=32, N=1, R=128, mcs=100, seed=1, tile=64, subsweeps=1),
    "C2": dict(L=1024, N=1, R=128, mcs=10_000, seed=1, tile=64, subsweeps=1),      # seeds 1..4
    "C3": dict(L=2048, N=1, R=64, mcs=5_000, seed=1, tile=64, subsweeps=1),        # N in 1..4
    "C4": dict(L=32768, N=1, R=1, mcs=2_000, seed=1, tile=64, subsweeps=1),
    "C5": dict(L=64, N=1, R=4096, mcs=15_521, seed=1, tile=64, subsweeps=4),       # L in 64..512, N in 1,2
    # not a BASELINE config: the paper's own largest system (L = 9605, t = 1e5 MCS, 128 realizations),
    # a lattice side that is not a power of two (general-L schedule), at 4 realizations
    "X1": dict(L=9605, N=1, R=4, mcs=100_000, seed=1, tile=64, subsweeps=1),
}


def c5_realizations(L):
    """BASELINE.json C5: 4096 realizations at L = 64, scaled as 1/L^2 (R * L^2 = 2^24)."""
    return (1 << 24) // (L * L)


def c5_mcs(L):
    """BASELINE.json C5: run to t = 20 * L^1.6 MCS."""
    return int(math.ceil(20.0 * L ** 1.6))


def log_spaced_times(t_max, n=64):
    """sorted(set(round(t_max^(j/(n-1))))) for j = 0..n-1: the `n log-spaced times` of C2-C4."""
    return sorted({int(round(t_max ** (j / (n - 1)))) for j in range(n)})


def eq10_times(t_max, m=0.01, t0=0.0):
    """The paper's measurement schedule, Eq. (10): t_{i+1} = (t_i + 10) e^m with m = 0.01, t_0 = 0.
    The recursion gives real numbers and the paper does not say how they are rounded (reading Q11): each t_i is
    rounded to the nearest integer MCS, duplicates are dropped, times beyond t_max are cut."""
    out, t = [], float(t0)
    while True:
        t = (t + 10.0) * math.exp(m)
        ti = int(round(t))
        if ti > t_max:
            break
        if not out or ti > out[-1]:
            out.append(ti)
    return out


def attempts(L, R, mcs):
    """1 MCS = L*L attempts per realization (reading Q4)."""
    return int(L) * int(L) * int(R) * int(mcs)


def replica_range(rank, world, r_per_gpu):
    """Multi-GPU = replicas only: rank i owns the global realizations
    [i * r_per_gpu, (i + 1) * r_per_gpu).  Returns (first_real, R) for rsos_init."""
    if not 0 <= rank < world:
        raise ValueError("rank %d outside [0, %d)" % (rank, world))
    return rank * int(r_per_gpu), int(r_per_gpu)
