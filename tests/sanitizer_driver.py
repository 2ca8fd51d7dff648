"""Short run of every kernel family, meant to be executed under compute-sanitizer on a B200:

    compute-sanitizer --tool memcheck|racecheck|synccheck python tests/sanitizer_driver.py

(`profiles/r02_sanitizer.md` records the results.)  `python tests/sanitizer_driver.py profile` is the short run that
`profiles/r02_ncu_small_and_observables.md` was taken from.  Not collected by pytest; it checks nothing itself except that
the runs finish and agree with each other where two kernels compute the same thing.
"""
import os
import sys

sys.path.insert(0, os.path.join(os.path.dirname(os.path.abspath(__file__)), ".."))
os.environ.setdefault("EA_RESIDENT_TIMEOUT_MS", "900000")  # the tools slow the flag waits of the persistent kernel down

import numpy as np  # noqa: E402

from paper_1411_5512_b200 import binding  # noqa: E402


def profile_run():
    """The short run behind profiles/r02_ncu_small_and_observables.md: SMALL at L = 8, 16, 32 (1000 sweeps each), then one
    measure point at L = 128."""
    for L, nrep in ((8, 1), (16, 2), (32, 2)):
        g = binding.Sim(L, 0.5, 0.8, n_replicas=nrep, seed=3, n_slots=1)
        g.sweep(1000)
        g.synchronize()
        g.close()
    g = binding.Sim(128, 0.77, 0.8, n_replicas=2, seed=3, n_slots=1)
    g.sweep(8); g.snapshot(0); g.sweep(8)
    g.autocorr(0); g.c4(64, with_q=True); g.energy(); g.magnetisation()
    g.close()


def main():
    if sys.argv[1:] == ["profile"]:
        return profile_run()
    which = sys.argv[1:] or ["resident", "rows", "fold", "observables", "c4vec", "batch"]
    if "resident" in which:  # persistent kernel: inter-CTA release/acquire flags, named barriers, mbarriers, cp.async
        a = binding.Sim(128, 0.77, 0.8, n_replicas=2, seed=7, n_slots=0, kernel="rows")
        b = binding.Sim(128, 0.77, 0.8, n_replicas=2, seed=7, n_slots=0, kernel="resident")
        a.sweep(3); b.sweep(3)
        assert np.array_equal(a.get_spins(), b.get_spins())
        a.close(); b.close()
        print("resident ok", flush=True)
    if "rows" in which:
        for kern in ("scalar", "vec2", "rows"):
            g = binding.Sim(16, 0.6, 0.8, n_replicas=2, seed=11, n_slots=1, kernel=kern)
            g.sweep(40)  # one graph replay + direct launches
            g.close()
        print("rows ok", flush=True)
    if "fold" in which:
        g = binding.Sim(16, 0.5, 0.8, n_replicas=2, seed=13, n_slots=0, n_samples=16)
        g.sweep(5)
        g.get_spins()
        g.close()
        print("fold ok", flush=True)
    if "observables" in which:
        for L in (16, 64):
            g = binding.Sim(L, 0.7, 0.8, n_replicas=2, seed=17, n_slots=1)
            g.sweep(2); g.snapshot(0); g.sweep(2)
            g.autocorr(0); g.c4(L // 2, with_q=True); g.energy(); g.magnetisation()
            g.close()
        print("observables ok", flush=True)
    if "c4vec" in which:
        g = binding.Sim(32, 0.7, 0.8, n_replicas=2, seed=19, n_slots=0)
        g.sweep(2)
        g.c4_shells(3)
        g.close()
        print("c4vec ok", flush=True)
    if "batch" in which:
        from paper_1411_5512_b200.scan import Scan
        sc = Scan([{"L": 16, "p": 0.5 + 0.1 * k, "T": 0.8, "seed": 23 + k} for k in range(4)])
        sc.sweep(40)
        sc.synchronize()
        sc.close()
        print("batch ok", flush=True)


if __name__ == "__main__":
    main()
