"""Seeded synthetic workloads: the BASELINE.json configurations and random input words.

This module holds NONE of the method's arithmetic (no Philox, no thresholds, no update
rule): it only names the paper's workload shapes (PAPER.md:98, :108 -- L up to 128,
T = 0.8, p in [0.5, 1], 64 samples per word, two replicas per disorder) and draws plain
numpy random words for tests that inject their own spins / bonds / gauge vectors.  It is
the one module both the oracle's tests and the CUDA path's tests/bench may import.

The paper's workloads are themselves synthetic (random +-J bonds, random start:
PAPER.md:25, :29), so a seeded (L, p, T, seed) tuple IS the paper's input distribution;
the lattice contents are drawn inside the library / the oracle from the written stream
definition.
"""
from dataclasses import dataclass

import numpy as np

SEED_BASE = 0x1411_5512_0000_0000  # + 0x100 * cfg + variant


@dataclass(frozen=True)
class Config:
    name: str
    L: int
    p: float
    T: float
    n_replicas: int      # 1: 64 independent samples, 2: 32 disorders x 2 replicas
    sweeps: int          # the run length BASELINE.json names
    seed: int
    parity_sweeps: int   # horizon checked bit-exactly against the oracle in tests

    @property
    def N(self):
        return self.L ** 3


def seed_for(cfg: int, variant: int = 0) -> int:
    return SEED_BASE + 0x100 * cfg + variant


# BASELINE.json "configs", in order.  cfg3 and cfg5 are small families (several p / T).
CONFIGS = {
    "cfg1": Config("cfg1", 8, 0.5, 0.8, 1, 1000, seed_for(1), 1000),
    "cfg2": Config("cfg2", 32, 0.5, 0.8, 2, 10 ** 5, seed_for(2), 3000),
    "cfg3a": Config("cfg3a", 64, 0.6, 0.8, 2, 10 ** 6, seed_for(3, 0), 300),
    "cfg3b": Config("cfg3b", 64, 0.7, 0.8, 2, 10 ** 6, seed_for(3, 1), 300),
    "cfg4": Config("cfg4", 128, 0.77, 0.8, 2, 10 ** 7, seed_for(4), 48),
    "cfg5_p0.5_T0.8": Config("cfg5_p0.5_T0.8", 128, 0.5, 0.8, 2, 10 ** 8, seed_for(5, 0), 8),
    "cfg5_p0.8_T0.8": Config("cfg5_p0.8_T0.8", 128, 0.8, 0.8, 2, 10 ** 8, seed_for(5, 1), 8),
    "cfg5_p0.9_T0.8": Config("cfg5_p0.9_T0.8", 128, 0.9, 0.8, 2, 10 ** 8, seed_for(5, 2), 8),
    "cfg5_p1.0_T0.8": Config("cfg5_p1.0_T0.8", 128, 1.0, 0.8, 2, 10 ** 8, seed_for(5, 3), 8),
    "cfg5_p0.5_T2.0": Config("cfg5_p0.5_T2.0", 128, 0.5, 2.0, 2, 10 ** 8, seed_for(5, 4), 8),
    "cfg5_p0.8_T2.0": Config("cfg5_p0.8_T2.0", 128, 0.8, 2.0, 2, 10 ** 8, seed_for(5, 5), 8),
    "cfg5_p0.9_T2.0": Config("cfg5_p0.9_T2.0", 128, 0.9, 2.0, 2, 10 ** 8, seed_for(5, 6), 8),
    "cfg5_p1.0_T2.0": Config("cfg5_p1.0_T2.0", 128, 1.0, 2.0, 2, 10 ** 8, seed_for(5, 7), 8),
}

BENCH_CONFIG = "cfg4"  # the L=128 workload BASELINE.json's metric / 70 % target is quoted on


def random_words(n: int, seed: int) -> np.ndarray:
    """n uniform 64-bit words (numpy PCG64)."""
    rng = np.random.default_rng(seed)
    return rng.integers(0, 2 ** 64, size=n, dtype=np.uint64)


def random_bond_words(N: int, p: float, n_replicas: int, seed: int) -> np.ndarray:
    """Canonical bond words [3*N]: bit = 1 (J = -1) with probability 1 - p, iid per bit
    (PAPER.md:25).  n_replicas == 2: lanes 32..63 repeat lanes 0..31."""
    rng = np.random.default_rng(seed)
    bits = rng.random((3 * N, 64)) >= p
    if n_replicas == 2:
        bits[:, 32:] = bits[:, :32]
    weights = (np.uint64(1) << np.arange(64, dtype=np.uint64))
    return (bits.astype(np.uint64) * weights).sum(axis=1, dtype=np.uint64)


def log_spaced_times(t_max: int, per_decade=(1, 2, 5)):
    """Measurement grid {1,2,5} x 10^m up to t_max."""
    out, m = [], 1
    while m <= t_max:
        for k in per_decade:
            if k * m <= t_max:
                out.append(k * m)
        m *= 10
    return out
