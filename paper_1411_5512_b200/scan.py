"""Scans: many independent sims advanced together ("temperature/p scans ... as a batched
multi-sim driver"; the paper's production is exactly that -- 192 samples = 3 batches of 64 at each of ~20 values of
p, and Delta p = 0.01 scans at L = 32 / 64, :134).

Small lattices cannot fill a B200 alone: one L = 64 half-sweep is a 256-CTA kernel that lasts 1.5 us behind a 2 us
launch.  Every `ea_sim` owns its own CUDA stream and its own CUDA graph, and distinct handles are independent
(include/ea.h), so K sims issued back to back overlap on the device: measured aggregate at L = 64, 32 x 2 replicas,
T = 0.8: 0.333 ps/attempt with 1 sim, 0.114 with 4, 0.078 with >= 8 (better than one L = 128 lattice).  This module
is only the dispatch loop and the bookkeeping; each point runs the same kernels through the same C ABI.

Across GPUs the points are dealt round-robin (replicas.shard): replicas only, no data-path collective.
"""
import numpy as np

from . import binding, replicas


class Scan:
    """points: iterable of dicts with keys L, p, T and optionally n_replicas (2), seed (0), n_slots (1), kernel."""

    def __init__(self, points, rank=0, world_size=1, device=None, fused="auto"):
        self.all_points = [dict(pt) for pt in points]
        self.index = replicas.shard(list(range(len(self.all_points))), rank, world_size)
        self.points = [self.all_points[k] for k in self.index]
        self.sims = []
        for pt in self.points:
            self.sims.append(binding.Sim(pt["L"], pt["p"], pt["T"], n_replicas=pt.get("n_replicas", 2),
                                         seed=pt.get("seed", 0), n_slots=pt.get("n_slots", 1),
                                         kernel=pt.get("kernel", "auto"), device=device))
        # Which points share launches (measured on B200, 2000-sweep calls, us per sweep of ALL points): none, unless asked.
        #   L <= 32: every point alone on its stream -- AUTO runs SMALL (lattice in the shared memory of one CTA / cluster, one
        #            launch per call): L = 16: 0.82 (16 points) / 1.41 (64) against 5.19 / 5.99 for the fused launches
        #            (ea_batch_*: one launch per colour for all points); L = 32: 3.9 / 13.1 / 24.9 with 16 / 64 / 128 points
        #            against 6.9 / 14.6 / 30.1 fused;
        #   L = 64:  streams of graph replays (10.2 for 8 points against 14 fused).
        # fused=True fuses every group of one shape (L in 16, 32, 64); "auto" and False do not.
        for s in self.sims:
            s.set_concurrency_hint(len(self.sims))   # many sims share the SMs: throughput-oriented code paths
        self.batches, self._solo = [], list(self.sims)
        groups = {}
        for s in self.sims:
            if s.n_samples == binding.LANES and s.L in (16, 32, 64):
                groups.setdefault((s.L, s.n_replicas), []).append(s)
        for (L, _), members in groups.items():
            if fused is True and len(members) > 1:
                self.batches.append(binding.Batch(members))
                self._solo = [s for s in self._solo if s not in members]

    def __len__(self):
        return len(self.sims)

    def sweep(self, n):
        """n sweeps of every point; asynchronous (each sim on its own stream), so the points overlap."""
        for b in self.batches:
            b.sweep(n)
        for s in self._solo:
            s.sweep(n)

    def synchronize(self):
        for s in self.sims:
            s.synchronize()

    def snapshot(self, slot=0):
        for s in self.sims:
            s.snapshot(slot)

    def measure(self, slot=None, r_max=None):
        """Per point: dict of the per-sample integer observables (E, M, and A for `slot`, B / q for r_max)."""
        out = []
        for s in self.sims:
            rec = s.measure(slot=slot, r_max=min(r_max, s.L // 2) if r_max is not None and s.n_replicas == 2 else None)
            rec["t"] = s.time
            out.append(rec)
        return out

    def gather(self, key, records):
        """[world, points_per_rank, ...] array of observable `key` (ranks own equally many points, or pad first)."""
        return replicas.gather_lanes(np.stack([np.asarray(r[key]) for r in records]))

    def close(self):
        for b in self.batches:
            b.close()
        self.batches = []
        for s in self.sims:
            s.close()
        self.sims = []
