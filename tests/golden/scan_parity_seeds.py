"""Choose the Philox keys of the trajectory-parity tests (tests/test_gpu_parity.py) with the ORACLE ALONE.

The fp32 CUDA path and the fp64 oracle take the same discontinuous decisions (accept tests, clock expiry, sampler
tests, ring and list edges, cell faces) only while none of them is closer to its threshold than the two paths differ
(R-17).  They differ by fp32 rounding of forces and velocities, which grows about linearly with the number of
steps (positions ~1e-7 A per step, relative velocity error likewise).  The oracle records the margin of every
decision; this script runs it for 100 steps in ten 10-step chunks and scores a seed by
    score = min over chunks k = 1..10 of  min(decision margin_k, 2 x list margin_k) / k,
i.e. how far, relative to the growing difference, its closest call was.  For every test configuration it prints the
seed with the LARGEST score in a fixed range (3000..3199): the most robust key by the oracle's own audit.  Nothing here
touches the CUDA path; the printed seeds are typed into the tests, which then assert event-log and trajectory parity
over the full 100 steps of BASELINE.json's north_star on them.

    python tests/golden/scan_parity_seeds.py [first last]
"""
import os
import sys

sys.path.insert(0, os.path.dirname(os.path.dirname(os.path.dirname(os.path.abspath(__file__)))))

from oracle import jump_oracle as jo
from paper_2412_15073_b200 import workloads as wl


def score(sysd, run, seed, chunks=10, call=None):
    o = jo.Oracle(sysd, **dict(run, seed=seed))
    s = float("inf")
    for k in range(1, chunks + 1):
        o.reset_stats()
        (call or (lambda oo: oo.jump_step(10)))(o)
        st = o.stats()
        s = min(s, min(st["min_margin"], 2.0 * st["min_list_margin"]) / k)
    o.close()
    return s


def best(name, sysd, run, first, last, **kw):
    sc = [(score(sysd, run, seed, **kw), seed) for seed in range(first, last)]
    sc.sort(reverse=True)
    print(name, "best seeds (score, seed):", [("%.2e" % a, b) for a, b in sc[:3]], flush=True)


if __name__ == "__main__":
    first, last = (int(sys.argv[1]), int(sys.argv[2])) if len(sys.argv) > 2 else (3000, 3200)
    sysd, run = wl.make_config(0)
    for eps, mode in ((1.0, 0), (0.3, 0), (float("inf"), 0), (2.0, 1)):
        r = dict(run, flags=3 | 4, eps_jump=eps, eps_mode=mode)
        best("jump_step x100 eps=%s mode=%d" % (eps, mode), sysd, r, first, last)
    best("bjaoajb x20", sysd, dict(run, flags=3 | 4 | 64), first, last, chunks=2)
    best("combined x100 (R-22)", sysd, dict(run, flags=3 | 4 | 128), first, last)
    for flags, mode in ((3, 0), (3 | 8, 0), (1, 0), (3, 1), (3 | 8, 1)):
        r = dict(run, flags=flags | 4, eps_mode=mode, eps_jump=2.0 if mode else run["eps_jump"])
        best("respa x3 flags=%d mode=%d" % (flags, mode), sysd, r, first, last, chunks=1, call=lambda o: o.jump_respa_step(3))
