"""A short tour of every update engine on small cases, checked against what holds for any correct run.

    python -m paper_1605_02620_b200.selfcheck [--mcs M] [--only NAME[,NAME...]] [--list]

For each case: rsos_init with an explicit engine (and lanes / cluster where the engine has them), rsos_advance, then every
read-out path (rsos_sums, rsos_width, rsos_moments, rsos_get_heights, rsos_sums_static) and three invariants the paper's
rule fixes (Eq. 6; P:79 flat start): heights never negative, sum h = accepted deposits, and |h(x) - h(x')| <= N
on every bond of the periodic lattice.  No oracle is involved (the bit-exact comparison lives in tests/); this module is
what a user runs to see that the library works on their GPU, and what `compute-sanitizer` is pointed at
(profiles/r3_sanitizer.md): every shared-memory kernel of the library is launched at least once, small enough for the
sanitizer's slowdown.  --repeat N runs every case N times and demands bit-identical heights each time (--noise: while a
second context keeps the GPU busy on another stream with a varying load), the check for results that depend on timing.
"""
import argparse
import hashlib
import sys

import numpy as np

from . import binding as B

# name -> (L, N, R, keyword arguments of Rsos, engine name rsos_info must report)
CASES = [
    ("thread_lanes1", 256, 1, 2, dict(engine=B.ENGINE_THREAD, lanes=1), "thread"),
    ("thread_lanes2", 256, 1, 2, dict(engine=B.ENGINE_THREAD, lanes=2), "thread"),
    ("thread_lanes4", 256, 1, 2, dict(engine=B.ENGINE_THREAD, lanes=4), "thread"),
    ("thread_lanes8", 256, 1, 2, dict(engine=B.ENGINE_THREAD, lanes=8), "thread"),
    ("thread_4bit_lanes4", 256, 3, 2, dict(engine=B.ENGINE_THREAD, lanes=4, subsweeps=2), "thread"),
    ("thread_general_L", 130, 1, 3, dict(), "thread"),
    ("resident_cluster1", 256, 1, 2, dict(engine=B.ENGINE_RESIDENT, subsweeps=4, cluster=1), "resident"),
    ("resident_cluster2", 512, 1, 1, dict(engine=B.ENGINE_RESIDENT, subsweeps=4, cluster=2), "resident"),
    ("resident_cluster4", 512, 2, 1, dict(engine=B.ENGINE_RESIDENT, subsweeps=4, cluster=4), "resident"),
    ("fine_8x8", 64, 1, 8, dict(engine=B.ENGINE_FINE, tile=8), "fine"),
    ("fine_16x16", 128, 2, 3, dict(engine=B.ENGINE_FINE, tile=16), "fine"),
    ("fine_poisson", 64, 1, 5, dict(tile=8, poisson=True), "fine"),
    ("level", 32, 1, 4, dict(engine=B.ENGINE_LEVEL), "level"),
    ("onchip", 32, 2, 9, dict(engine=B.ENGINE_ONCHIP), "onchip"),
    ("multi", 32, 1, 128, dict(multisurface=True), "multi"),
    ("warp", 256, 5, 2, dict(engine=B.ENGINE_WARP), "warp"),
    ("simple_window_general_L", 150, 1, 2, dict(engine=B.ENGINE_SIMPLE), "simple"),
    ("simple_global", 128, 40, 1, dict(engine=B.ENGINE_SIMPLE), "simple"),
]


def run_case(name, L, N, R, kw, engine, mcs):
    import torch
    g = B.Rsos(L, N, R, 11, **kw)
    info = g.info()
    if info["engine"] != engine:
        raise AssertionError("%s: engine %s, expected %s" % (name, info["engine"], engine))
    g.advance(mcs)
    s1, s2, acc = g.sums()
    g.advance(1)                                           # a second call: engines that keep state on chip reload it
    s1, s2, acc = g.sums()
    w2, hm = g.width()
    base, M = g.moments()
    h = g.heights().astype(np.int64)
    if h.min() < 0:
        raise AssertionError("%s: negative height" % name)
    if not (h.sum(axis=(1, 2)) == s1).all() or not ((h * h).sum(axis=(1, 2)).astype(np.uint64) == s2).all():
        raise AssertionError("%s: rsos_sums disagrees with the heights" % name)
    if not (s1 == acc).all():
        raise AssertionError("%s: sum h != accepted deposits" % name)
    for ax in (1, 2):
        if np.abs(h - np.roll(h, 1, axis=ax)).max() > N:
            raise AssertionError("%s: Eq. (6) violated" % name)
    for r in range(R):
        if M[r][0] != int(s1[r]) - int(base[r]) * L * L:
            raise AssertionError("%s: first power sum" % name)
    # the allocation-free sums on the same surfaces
    if R <= B.STATIC_MAX_R:
        o1 = torch.zeros(R, dtype=torch.int64, device="cuda")
        o2 = torch.zeros(R, dtype=torch.int64, device="cuda")
        B.sums_static(g.device_heights(), L, R, o1.data_ptr(), o2.data_ptr(), None)
        torch.cuda.synchronize()
        if not (o1.cpu().numpy() == s1).all() or not (o2.cpu().numpy().view(np.uint64) == s2).all():
            raise AssertionError("%s: rsos_sums_static disagrees with rsos_sums" % name)
    digest = hashlib.sha256(h.tobytes()).hexdigest()
    g.close()
    return {"case": name, "digest": digest, "engine": info["engine"], "lanes": info["lanes"], "cluster": info["cluster"], "bits": info["packed_bits"],
            "hmean": float(hm.mean()), "W2": float(w2.mean())}


def main(argv=None):
    ap = argparse.ArgumentParser()
    ap.add_argument("--mcs", type=int, default=2)
    ap.add_argument("--only", default="")
    ap.add_argument("--list", action="store_true")
    ap.add_argument("--repeat", type=int, default=1, help="run every case this many times; all heights must be identical")
    ap.add_argument("--noise", action="store_true", help="with --repeat: another context advances on a second stream meanwhile")
    a = ap.parse_args(argv)
    if a.list:
        print("\n".join(c[0] for c in CASES))
        return 0
    only = set(filter(None, a.only.split(",")))
    import torch
    if not torch.cuda.is_available():
        raise SystemExit("selfcheck: no CUDA device (the library has no CPU fallback)")
    noise = None
    if a.noise:                                            # a second context on its own stream keeps the GPU busy meanwhile
        noise_stream = torch.cuda.Stream()
        noise = B.Rsos(2048, 1, 8, 99, stream=noise_stream.cuda_stream)
    for name, L, N, R, kw, engine in CASES:
        if only and name not in only:
            continue
        out = run_case(name, L, N, R, kw, engine, a.mcs)
        for i in range(1, a.repeat):
            if noise:
                noise.advance(1 + i % 3)                   # asynchronous: overlaps the case below with a varying load
            again = run_case(name, L, N, R, kw, engine, a.mcs)
            if again["digest"] != out["digest"]:
                raise AssertionError("%s: repeat %d gave different heights (a timing-dependent result)" % (name, i))
        print("ok  %-26s engine=%-8s lanes=%-2d cluster=%-2d bits=%d  <h>=%.3f  W2=%.4f  runs=%d sha256=%s" % (
            out["case"], out["engine"], out["lanes"], out["cluster"], out["bits"], out["hmean"], out["W2"], max(1, a.repeat),
            out["digest"][:12]), flush=True)
    if noise:
        noise.close()
    return 0


if __name__ == "__main__":
    sys.exit(main())
