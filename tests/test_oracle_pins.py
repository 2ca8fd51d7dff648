"""Pins of the CPU oracle against what the paper and the mathematics fix (no GPU).

Every pin is chosen so that a plausible mistake in oracle/ea_oracle.c -- a dropped bond, a
wrong sign, a factor in the Boltzmann exponent, a swapped lane/half mapping, a transposed
index -- fails at least one of them.  Pin numbers P1..P13 follow SURVEY.md section 8(c).
Citations are PAPER.md:<line>.
"""
import itertools
import math
import os

import numpy as np
import pytest

import oracle
from oracle import Oracle
from paper_1411_5512_b200 import workloads as wl

GOLDEN = os.path.join(os.path.dirname(__file__), "golden")
ALL = np.uint64(0xFFFFFFFFFFFFFFFF)


# ----------------------------------------------------------------------------------------
# independent numpy helpers (no oracle code): unpack, brute-force energy
# ----------------------------------------------------------------------------------------
def unpack(words, n_lanes=64):
    """uint64 words [n] -> +-1 int array [n_lanes][n], bit 1 <-> -1 (contract C-A2)."""
    w = np.asarray(words, dtype=np.uint64)
    bits = (w[None, :] >> np.arange(n_lanes, dtype=np.uint64)[:, None]) & np.uint64(1)
    return 1 - 2 * bits.astype(np.int64)


def energy_numpy(S, J, L):
    """H = -sum_<ij> J_ij S_i S_j (Eq. 1) with np.roll; S [lanes][N], J [lanes][3][N]."""
    lanes = S.shape[0]
    S3 = S.reshape(lanes, L, L, L)          # [lane][z][y][x]
    E = np.zeros(lanes, dtype=np.int64)
    for d, axis in ((0, 3), (1, 2), (2, 1)):
        Jd = J[:, d, :].reshape(lanes, L, L, L)
        E -= (Jd * S3 * np.roll(S3, -1, axis=axis)).sum(axis=(1, 2, 3))
    return E


# ----------------------------------------------------------------------------------------
# P1  Philox4x32-10 block function: published known-answer vectors
# ----------------------------------------------------------------------------------------
def test_P1_philox_known_answers():
    n = 0
    for line in open(os.path.join(GOLDEN, "philox4x32_10_kat.txt")):
        if line.startswith("#") or not line.strip():
            continue
        lhs, rhs = line.split("->")
        v = [int(x, 16) for x in lhs.split()]
        want = [int(x, 16) for x in rhs.split()]
        got = oracle.philox4x32_10(v[:4], v[4:6])
        assert [int(x) for x in got] == want
        n += 1
    assert n == 3


def test_P1b_philox_is_a_bijection_on_a_small_slice():
    # a counter-based generator is a keyed bijection: distinct counters -> distinct blocks
    outs = {tuple(int(x) for x in oracle.philox4x32_10([i, 7, 0, 1], [3, 4])) for i in range(2000)}
    assert len(outs) == 2000


# ----------------------------------------------------------------------------------------
# P3  thresholds (closed form) and the single-spin decision (Eq. 9)
# ----------------------------------------------------------------------------------------
def test_P3_thresholds_golden_and_closed_form():
    for line in open(os.path.join(GOLDEN, "thresholds.txt")):
        if line.startswith("#") or not line.strip():
            continue
        f = line.split()
        T = float(f[0])
        assert [int(x) for x in oracle.thresholds(T)] == [int(x) for x in f[1:4]]
    for T in (0.3, 0.8, 1.102, 2.0, 4.5115, 50.0):
        thr = oracle.thresholds(T)
        for n_u in range(3):
            local_sum = 6 - 2 * n_u
            p_eq9 = min(1.0, math.exp(-(2.0 / T) * local_sum))   # Eq. 9 verbatim
            assert abs(int(thr[n_u]) / 2.0 ** 32 - p_eq9) <= 2.0 ** -33 + 1e-18


def test_P3_single_spin_decision_at_the_threshold_edges():
    for T in (0.8, 2.0):
        thr = oracle.thresholds(T)
        for local_sum in (-6, -4, -2, 0):               # Delta E <= 0: always (incl. Delta E = 0)
            for r in (0, 1, 12345, 2 ** 32 - 1):
                assert oracle.accept(thr, local_sum, r)
        for n_u, local_sum in ((0, 6), (1, 4), (2, 2)):
            t = int(thr[n_u])
            assert oracle.accept(thr, local_sum, t - 1)
            assert not oracle.accept(thr, local_sum, t)
            assert not oracle.accept(thr, local_sum, 2 ** 32 - 1)
            assert oracle.accept(thr, local_sum, 0)
    thr0 = oracle.thresholds(0.0)
    assert not any(oracle.accept(thr0, s, 0) for s in (2, 4, 6))
    thr_inf = oracle.thresholds(float("inf"))
    assert all(oracle.accept(thr_inf, s, 2 ** 32 - 1) for s in (2, 4, 6))


def test_P3_acceptance_frequency_with_frozen_neighbours():
    # p = 1, all spins up: every spin has n_u = 0, so after ONE half-sweep the flipped fraction of the
    # colour must be thr[0] / 2^32 = exp(-12/T) within binomial error.  T = 6 -> 0.1353.
    L, T = 16, 6.0
    o = Oracle(L, 1.0, T, 1, seed=99)
    o.set_spins(np.zeros(o.N, dtype=np.uint64))
    o.half_sweep(0)
    S = o.spin_bytes()
    n_colour = o.N // 2
    # lanes 0..31 share one random number per site, lanes 32..63 another: two independent binomials
    for lane in (0, 31, 32, 63):
        flipped = int((S[lane] < 0).sum())
        pr = math.exp(-12.0 / T)
        assert abs(flipped - n_colour * pr) < 5 * math.sqrt(n_colour * pr * (1 - pr))
    assert (S[0] == S[31]).all() and (S[32] == S[63]).all()   # shared number, same environment
    assert (S[0] != S[32]).any()                             # the halves do not share it (C-A7)


# ----------------------------------------------------------------------------------------
# stream layout (C-A6, C-A7): same-colour sites j = x >> 1 of an x-row pair up (j even, j + 1); the pair shares the
# block at counter (first site, t lo, t hi, tag); first site: out[0] -> lanes 0..31, out[1] -> 32..63; second
# site: out[2], out[3].  L = 6 has an unpaired last site per row (L/2 odd), L = 2 only single sites.
# ----------------------------------------------------------------------------------------
@pytest.mark.parametrize("L", [2, 4, 6, 8])
def test_stream_layout_of_update_numbers(L):
    T, seed = 6.0, 0xABCDEF0123456789
    key = [seed & 0xFFFFFFFF, seed >> 32]
    thr0 = int(oracle.thresholds(T)[0])
    for t in (0, 5, (1 << 32) + 3):
        for parity in (0, 1):
            o = Oracle(L, 1.0, T, 1, seed=seed)
            o.set_spins(np.zeros(o.N, dtype=np.uint64))   # all up, p = 1: n_u = 0 everywhere
            o.time = t
            o.half_sweep(parity)
            w = o.get_spins()
            for site in range(o.N):
                x, y, z = site % L, (site // L) % L, site // (L * L)
                if (x + y + z) & 1 != parity:
                    assert w[site] == 0
                    continue
                second = (x >> 1) & 1
                first_site = site - 2 * second
                out = oracle.philox4x32_10([first_site, t & 0xFFFFFFFF, t >> 32, parity], key)
                lo = 0xFFFFFFFF if int(out[2 * second]) < thr0 else 0
                hi = 0xFFFFFFFF if int(out[2 * second + 1]) < thr0 else 0
                assert int(w[site]) == lo | (hi << 32)


def test_stream_layout_of_init():
    L, seed = 4, 0x0123456789ABCDEF
    key = [seed & 0xFFFFFFFF, seed >> 32]
    for n_rep in (1, 2):
        o = Oracle(L, 0.3, 0.8, n_rep, seed=seed)
        w, b = o.get_spins(), o.get_bonds()
        P = int(round(2 ** 32 * 0.3))
        assert oracle.bond_threshold(0.3) == P
        for site in (0, 1, 17, o.N - 1):
            out = oracle.philox4x32_10([site, 0, 0, 2], key)
            assert int(w[site]) == int(out[0]) | (int(out[1]) << 32)
            for d in range(3):
                word = 0
                for lane in range(64 if n_rep == 1 else 32):
                    out = oracle.philox4x32_10([site, 16 * d + (lane >> 2), 0, 3], key)
                    if not int(out[lane & 3]) < P:
                        word |= 1 << lane
                if n_rep == 2:
                    word |= word << 32
                assert int(b[d * o.N + site]) == word


# ----------------------------------------------------------------------------------------
# P2  exact Boltzmann statistics on L = 2 by brute force (2^8 states)
# ----------------------------------------------------------------------------------------
def _l2_energies(Jlane):
    """All 256 energies of one L=2 sample from Eq. 1; Jlane [3][8] of +-1.  On L=2 the +x and -x
    neighbours coincide and the two forward bonds between a pair are distinct bonds (C-S15)."""
    L = 2
    E = np.zeros(256)
    for state in range(256):
        S = np.array([1 - 2 * ((state >> i) & 1) for i in range(8)])
        e = 0
        for site in range(8):
            x, y, z = site % L, (site // L) % L, site // (L * L)
            nb = [((x + 1) % L) + L * (y + L * z), x + L * (((y + 1) % L) + L * z), x + L * (y + L * ((z + 1) % L))]
            for d in range(3):
                e -= Jlane[d][site] * S[site] * S[nb[d]]
        E[state] = e
    return E


def test_P2_metropolis_rule_with_integer_thresholds_leaves_boltzmann_stationary():
    # exact 256x256 matrix of one half-sweep built from thr/2^32; pi P = pi up to the 2^-33 rounding of
    # the thresholds.  (This pins the READING C-A4, independent of the oracle's code.)
    T = 2.0
    rng = np.random.default_rng(5)
    J = rng.choice([-1, 1], size=(3, 8))
    E = _l2_energies(J)
    pi = np.exp(-E / T)
    pi /= pi.sum()
    thr = [int(x) / 2.0 ** 32 for x in oracle.thresholds(T)]
    L = 2

    def local_sum(S, site):
        x, y, z = site % L, (site // L) % L, site // (L * L)
        s = 0
        for d, (dx, dy, dz) in enumerate(((1, 0, 0), (0, 1, 0), (0, 0, 1))):
            f = ((x + dx) % L) + L * (((y + dy) % L) + L * ((z + dz) % L))
            b = ((x - dx) % L) + L * (((y - dy) % L) + L * ((z - dz) % L))
            s += J[d][site] * S[site] * S[f] + J[d][b] * S[site] * S[b]
        return s

    for parity in (0, 1):
        sites = [s for s in range(8) if ((s % 2) + ((s // 2) % 2) + (s // 4)) % 2 == parity]
        P = np.zeros((256, 256))
        for state in range(256):
            S = np.array([1 - 2 * ((state >> i) & 1) for i in range(8)])
            pf = []
            for s in sites:
                ls = local_sum(S, s)
                pf.append(1.0 if ls <= 0 else thr[(6 - ls) // 2])
            for flips in itertools.product((0, 1), repeat=4):
                pr, new = 1.0, state
                for s, f, q in zip(sites, flips, pf):
                    pr *= q if f else 1 - q
                    if f:
                        new ^= 1 << s
                P[state, new] += pr
        assert np.abs(pi @ P - pi).max() < 1e-8


def _l2_sweep_matrix(J, T, rule="metropolis"):
    """Exact 256x256 transition matrix of one sweep (parity 0 then 1) of checkerboard dynamics on L = 2,
    built ONLY from the brute-force energies: Metropolis a(s -> s^i) = min(1, exp(-(E(s^i) - E(s)) / T)) (Eq. 9),
    heat bath a = 1 / (1 + exp((E(s^i) - E(s)) / T)) (C-HB)."""
    E = _l2_energies(J)
    P_full = np.eye(256)
    for parity in (0, 1):
        sites = [s for s in range(8) if ((s % 2) + ((s // 2) % 2) + (s // 4)) % 2 == parity]
        P = np.zeros((256, 256))
        for state in range(256):
            if rule == "metropolis":
                acc = [min(1.0, math.exp(-(E[state ^ (1 << s)] - E[state]) / T)) for s in sites]
            else:
                acc = [1.0 / (1.0 + math.exp((E[state ^ (1 << s)] - E[state]) / T)) for s in sites]
            for flips in itertools.product((0, 1), repeat=4):
                pr, new = 1.0, state
                for s, f, q in zip(sites, flips, acc):
                    pr *= q if f else 1 - q
                    if f:
                        new ^= 1 << s
                P[state, new] += pr
        P_full = P_full @ P
    return E, P_full


@pytest.mark.parametrize("rule", ["metropolis", "heatbath"])
def test_P2_oracle_one_sweep_transitions_match_the_exact_boltzmann_metropolis_matrix(rule):
    # For EVERY one of the 256 states, the oracle's empirical next-state distribution after one sweep
    # (over many sweep counters t = independent random numbers) must equal the exact row of the matrix
    # above, and that matrix must leave exp(-H/T)/Z stationary (detailed balance per half-sweep).
    T, K = 2.0, 1500
    o = Oracle(2, 0.5, T, 1, seed=77)
    o.set_dynamics(rule)
    rng = np.random.default_rng(12)
    J = rng.choice([-1, 1], size=(3, 8))
    o.set_bonds(np.where(J.reshape(-1) < 0, ALL, np.uint64(0)))           # same disorder in all 64 lanes
    E, P = _l2_sweep_matrix(J, T, rule)
    pi = np.exp(-E / T)
    pi /= pi.sum()
    assert np.abs(pi @ P - pi).max() < 1e-12                              # Boltzmann is stationary
    weights = (1 << np.arange(8)).astype(np.int64)
    lanes = np.arange(64, dtype=np.uint64)
    chi2, dof, zmax = 0.0, 0, 0.0
    for batch in range(4):                                                # lane b starts in state 64*batch + b
        start = 64 * batch + np.arange(64)
        words = np.zeros(8, dtype=np.uint64)
        for site in range(8):
            words[site] = (((start >> site) & 1).astype(np.uint64) << lanes).sum(dtype=np.uint64)
        hist = np.zeros((64, 256))
        for t in range(K):
            o.set_spins(words)
            o.time = 1000 * batch + t
            o.sweep(1)
            nxt = ((o.spin_bytes() < 0).astype(np.int64) * weights[None, :]).sum(axis=1)
            hist[np.arange(64), nxt] += 1
        for b in range(64):
            exp = K * P[start[b]]
            assert hist[b][exp == 0].sum() == 0                           # impossible moves never happen
            big = exp >= 8
            ob = np.append(hist[b][big], hist[b][~big].sum())
            ex = np.append(exp[big], exp[~big].sum())
            keep = ex > 0
            chi2 += (((ob - ex) ** 2)[keep] / ex[keep]).sum()
            dof += int(keep.sum()) - 1
            # per-site flip marginals as z-scores
            for site in range(8):
                pf = P[start[b]][[(s ^ start[b]) >> site & 1 == 1 for s in range(256)]].sum()
                nf = hist[b][[(s ^ start[b]) >> site & 1 == 1 for s in range(256)]].sum()
                if 1e-9 < pf < 1 - 1e-9:
                    zmax = max(zmax, abs(nf - K * pf) / math.sqrt(K * pf * (1 - pf)))
                else:
                    assert nf == round(K * pf)                            # certain / impossible flips
    assert 0.85 * dof < chi2 < 1.15 * dof, (chi2, dof)
    assert zmax < 5.0, zmax
    # power: the same data against a matrix with a 10 % wrong temperature is rejected
    _, Pbad = _l2_sweep_matrix(J, 1.1 * T)
    assert np.abs(Pbad - P).max() > 0.01


def test_P2_long_run_histogram_of_the_L2_ferromagnet_is_boltzmann():
    T, sweeps = 3.0, 30000
    o = Oracle(2, 1.0, T, 1, seed=5)
    E = _l2_energies(np.ones((3, 8), dtype=np.int64))
    pi = np.exp(-E / T)
    pi /= pi.sum()
    weights = (1 << np.arange(8)).astype(np.int64)
    hist = np.zeros((2, 256))
    S = o.spin_bytes()
    o.sweep(50)
    for _ in range(sweeps):
        o.sweep(1)
        for k, lane in enumerate((0, 32)):                                # one lane per random-number half
            hist[k, int(((S[lane] < 0) * weights).sum())] += 1
    for k in range(2):
        assert 0.5 * np.abs(hist[k] / sweeps - pi).sum() < 0.05           # total-variation distance
    pi_bad = np.exp(-E / (1.25 * T))
    pi_bad /= pi_bad.sum()
    assert 0.5 * np.abs(pi_bad - pi).sum() > 0.15                         # what a wrong exponent would give


# ----------------------------------------------------------------------------------------
# P4 / P5 / P6 / P8: energy bookkeeping, T = 0, p = 1, T = inf
# ----------------------------------------------------------------------------------------
@pytest.mark.parametrize("L,n_rep", [(2, 1), (4, 2), (6, 1), (8, 2)])
def test_P4_energy_from_eq1_equals_accumulated_delta_e(L, n_rep):
    o = Oracle(L, 0.6, 1.3, n_rep, seed=L)
    E0 = o.energy()
    for _ in range(12):
        o.sweep(1)
        assert (o.energy() - E0 == o.dE_accum()).all()
    # and energy() itself against the numpy-roll restatement of Eq. 1
    assert (o.energy() == energy_numpy(o.spin_bytes().astype(np.int64), o.bond_bytes().astype(np.int64), L)).all()


def test_P5_zero_temperature_never_raises_the_energy():
    o = Oracle(6, 0.5, 0.0, 1, seed=3)
    assert [int(x) for x in o.thresholds] == [0, 0, 0]
    E = o.energy()
    for _ in range(25):
        o.half_sweep(0)
        E1 = o.energy()
        assert (E1 <= E).all()
        o.half_sweep(1)
        E2 = o.energy()
        assert (E2 <= E1).all()
        E = E2
    assert (E < Oracle(6, 0.5, 0.0, 1, seed=3).energy()).all()      # and it did relax


def test_P6_ferromagnet_ground_state():
    for L in (2, 4, 8):
        o = Oracle(L, 1.0, 0.0, 1, seed=11)
        assert (o.bond_bytes() == 1).all()                           # p = 1: Ising ferromagnet
        o.set_spins(np.zeros(o.N, dtype=np.uint64))
        assert (o.energy() == -3 * o.N).all() and (o.magnetisation() == o.N).all()
        o.sweep(3)                                                   # T = 0: fixed point
        assert (o.get_spins() == 0).all()
        o.set_spins(np.full(o.N, ALL, dtype=np.uint64))              # all down: same energy, M = -N
        assert (o.energy() == -3 * o.N).all() and (o.magnetisation() == -o.N).all()
    o = Oracle(4, 0.0, 0.8, 1, seed=11)
    assert (o.bond_bytes() == -1).all()                              # p = 0: all antiferromagnetic


def test_P8_infinite_temperature_flips_everything_every_sweep():
    o = Oracle(4, 0.5, float("inf"), 2, seed=8)
    w0 = o.get_spins()
    o.snapshot(0)
    for t in range(1, 6):
        o.sweep(1)
        assert (o.get_spins() == (w0 ^ ALL if t & 1 else w0)).all()
        assert (o.autocorr(0) == (-o.N if t & 1 else o.N)).all()     # C(t, 0) = (-1)^t


# ----------------------------------------------------------------------------------------
# P7  exact gauge equivalence  S_i -> eps_i S_i,  J_ij -> eps_i eps_j J_ij
# ----------------------------------------------------------------------------------------
@pytest.mark.parametrize("L", [2, 4, 6])
def test_P7_gauge_transformation_commutes_with_the_dynamics(L):
    N, seed = L ** 3, 77
    a = Oracle(L, 0.5, 0.9, 1, seed=seed)
    b = Oracle(L, 0.5, 0.9, 1, seed=seed)
    eps = wl.random_words(N, 4242)
    idx = np.arange(N)
    x, y, z = idx % L, (idx // L) % L, idx // (L * L)
    fwd = [((x + 1) % L) + L * (y + L * z), x + L * (((y + 1) % L) + L * z), x + L * (y + L * ((z + 1) % L))]
    bonds = a.get_bonds().reshape(3, N)
    b.set_spins(a.get_spins() ^ eps)
    b.set_bonds(np.stack([bonds[d] ^ eps ^ eps[fwd[d]] for d in range(3)]).reshape(-1))
    assert (a.energy() == b.energy()).all()
    for _ in range(30):
        a.sweep(1)
        b.sweep(1)
        assert (b.get_spins() == a.get_spins() ^ eps).all()
    assert (a.get_spins() != Oracle(L, 0.5, 0.9, 1, seed=seed).get_spins()).any()   # something moved


# ----------------------------------------------------------------------------------------
# P9 / P10 / P13: order, lane independence, composition and resume
# ----------------------------------------------------------------------------------------
def test_P9_visiting_order_within_a_colour_is_immaterial():
    ref = Oracle(4, 0.5, 1.0, 1, seed=5)
    ref.sweep(10)
    for order in (1, 2):
        o = Oracle(4, 0.5, 1.0, 1, seed=5)
        o.set_order(order)
        o.sweep(10)
        assert (o.get_spins() == ref.get_spins()).all()
    o = Oracle(6, 0.5, 1.0, 1, seed=5)       # N not a power of two: the other shuffle branch
    o2 = Oracle(6, 0.5, 1.0, 1, seed=5)
    o2.set_order(2)
    o.sweep(5), o2.sweep(5)
    assert (o.get_spins() == o2.get_spins()).all()


def _permute_lanes(words, perm):
    w = np.asarray(words, dtype=np.uint64)
    out = np.zeros_like(w)
    for src, dst in enumerate(perm):
        out |= ((w >> np.uint64(src)) & np.uint64(1)) << np.uint64(dst)
    return out


def test_P10_lanes_are_independent_and_halves_own_their_random_number():
    L, seed = 4, 21
    rng = np.random.default_rng(0)
    perm = list(rng.permutation(32)) + [32 + int(v) for v in rng.permutation(32)]   # within halves
    a = Oracle(L, 0.5, 1.2, 1, seed=seed)
    b = Oracle(L, 0.5, 1.2, 1, seed=seed)
    b.set_spins(_permute_lanes(a.get_spins(), perm))
    b.set_bonds(_permute_lanes(a.get_bonds(), perm))
    a.sweep(15), b.sweep(15)
    assert (b.get_spins() == _permute_lanes(a.get_spins(), perm)).all()
    # swapping the two halves is NOT a symmetry (they use different random numbers)
    swap = [(i + 32) % 64 for i in range(64)]
    c = Oracle(L, 0.5, 1.2, 1, seed=seed)
    ref = Oracle(L, 0.5, 1.2, 1, seed=seed)
    c.set_spins(_permute_lanes(ref.get_spins(), swap))
    c.set_bonds(_permute_lanes(ref.get_bonds(), swap))
    c.sweep(15), ref.sweep(15)
    assert (c.get_spins() != _permute_lanes(ref.get_spins(), swap)).any()
    # a lane does not see the others: zero every other lane's spins and bonds, lane 5 is unchanged
    d = Oracle(L, 0.5, 1.2, 1, seed=seed)
    e = Oracle(L, 0.5, 1.2, 1, seed=seed)
    m = np.uint64(1 << 5)
    e.set_spins(d.get_spins() & m)
    e.set_bonds(d.get_bonds() & m)
    d.sweep(15), e.sweep(15)
    assert ((d.get_spins() & m) == (e.get_spins() & m)).all()


def test_P13_composition_and_resume():
    a = Oracle(4, 0.5, 0.8, 2, seed=9)
    a.sweep(10)
    b = Oracle(4, 0.5, 0.8, 2, seed=9)
    b.sweep(4)
    saved, t = b.get_spins(), b.time
    c = Oracle(4, 0.9, 0.8, 2, seed=1234)          # a different sim restored from the checkpoint
    c.set_bonds(b.get_bonds())
    c.set_spins(saved)
    c.time = t
    # the stream is keyed by the seed: restoring into another seed must NOT reproduce ...
    c.sweep(6)
    assert (c.get_spins() != a.get_spins()).any()
    # ... restoring into the same seed must
    d = Oracle(4, 0.5, 0.8, 2, seed=9)
    d.set_spins(saved)
    d.time = t
    d.sweep(6)
    assert (d.get_spins() == a.get_spins()).all() and d.time == 10


# ----------------------------------------------------------------------------------------
# P11  observables against numpy / FFT restatements and their special cases
# ----------------------------------------------------------------------------------------
def test_P11_observables_against_numpy_and_fft():
    L = 8
    o = Oracle(L, 0.5, 0.8, 2, seed=31)
    o.sweep(3)
    o.snapshot(0)
    W = unpack(o.get_spins())
    assert (unpack(o.get_snapshot(0)) == W).all()
    assert (o.autocorr(0) == o.N).all()                                    # A(t = 0) = N
    o.sweep(7)
    S = unpack(o.get_spins())
    assert (S == o.spin_bytes()).all()                                     # packed format <-> bytes
    assert (o.autocorr(0) == (W * S).sum(axis=1)).all()                    # Eq. 7
    assert (o.magnetisation() == S.sum(axis=1)).all()
    J = unpack(o.get_bonds()).reshape(64, 3, o.N)
    assert (J == o.bond_bytes()).all()
    assert (o.energy() == energy_numpy(S, J, L)).all()                     # Eq. 1
    q = S[:32] * S[32:]                                                    # Eq. 2
    assert (o.overlap() == q.sum(axis=1)).all()
    B = o.c4(L // 2)
    q3 = q.reshape(32, L, L, L).astype(np.float64)                         # [b][z][y][x]
    for d, axis in ((0, 3), (1, 2), (2, 1)):
        F = np.fft.fft(q3, axis=axis)
        corr = np.fft.ifft(F * np.conj(F), axis=axis).real                 # circular autocorrelation per line
        other = tuple(a for a in (1, 2, 3) if a != axis)
        tot = np.rint(corr.sum(axis=other)).astype(np.int64)               # [b][r], r = 0..L-1
        assert (B[d] == tot[:, : L // 2 + 1].T).all()                      # Eq. 3 along axis d
        for r in range(1, L // 2):
            assert (o.c4_one(d, L - r) == B[d][r]).all()                   # B(d, r) = B(d, L - r)
        assert (B[d][0] == o.N).all()                                      # B(d, 0) = N
        lines = q3.sum(axis=axis)                                          # sum_r B(d, r) = sum_lines (sum q)^2
        full = sum(o.c4_one(d, r) for r in range(L))
        assert (full == np.rint((lines ** 2).sum(axis=(1, 2))).astype(np.int64)).all()


def test_P11_identical_replicas_give_full_correlation():
    o = Oracle(4, 0.5, 0.8, 2, seed=1)
    w = o.get_spins()
    lo = w & np.uint64(0xFFFFFFFF)
    o.set_spins(lo | (lo << np.uint64(32)))
    assert (o.overlap() == o.N).all() and (o.c4(2) == o.N).all()
    with pytest.raises(ValueError):
        Oracle(4, 0.5, 0.8, 1, seed=1).c4(2)                              # needs two replicas


# ----------------------------------------------------------------------------------------
# P16  heat-bath variant (reading C-HB) -- not the paper's dynamics
# ----------------------------------------------------------------------------------------
def test_P16_heatbath_thresholds_closed_form_symmetry_and_limits():
    for T in (0.5, 0.8, 2.0, 7.3):
        thr = [int(x) for x in oracle.thresholds_heatbath(T)]
        for n_u in range(7):
            dE = 12 - 4 * n_u
            assert abs(thr[n_u] / 2.0 ** 32 - 1.0 / (1.0 + math.exp(dE / T))) <= 2.0 ** -32   # closed form
            assert abs(thr[n_u] + thr[6 - n_u] - 2 ** 32) <= 1                                 # P(dE) + P(-dE) = 1
        assert thr[3] == 2 ** 31 and thr == sorted(thr)                                        # dE = 0: exactly 1/2
        m = [int(x) for x in oracle.thresholds(T)]                                             # detailed balance ratio
        for n_u in range(3):                                                                   # P(dE)/P(-dE) = e^{-dE/T} = Metropolis
            assert abs(thr[n_u] / thr[6 - n_u] - m[n_u] / 2.0 ** 32) < 1e-6 * max(1.0, m[n_u] / 2.0 ** 32) + 2e-9
    assert [int(x) for x in oracle.thresholds_heatbath(0.0)] == [0, 0, 0, 2 ** 31, 2 ** 32, 2 ** 32, 2 ** 32]
    assert [int(x) for x in oracle.thresholds_heatbath(float("inf"))] == [2 ** 31] * 7
    thr = oracle.thresholds_heatbath(0.8)
    for n_u in range(7):                                                                       # strict "<" at the edge
        t = int(thr[n_u])
        if 0 < t < 2 ** 32:
            assert oracle.accept_heatbath(thr, 6 - 2 * n_u, t - 1) and not oracle.accept_heatbath(thr, 6 - 2 * n_u, t)


def test_P16_heatbath_single_spin_frequencies_and_energy_bookkeeping():
    L, T = 4, 6.0
    o = Oracle(L, 1.0, T, 1, seed=5)
    o.set_dynamics("heatbath")
    K, flips = 600, np.zeros(64)
    for t in range(K):                                    # all-up ferromagnet: n_u = 0 at every site, P = 1/(1+e^{12/T})
        o.set_spins(np.zeros(o.N, dtype=np.uint64))
        o.time = t
        o.half_sweep(0)
        flips += (o.spin_bytes() < 0).sum(axis=1)
    pf = 1.0 / (1.0 + math.exp(12.0 / T))
    n = K * o.N // 2
    assert abs(flips.sum() / 64 - n * pf) < 5 * math.sqrt(n * pf * (1 - pf) / 2)   # the 64 lanes share 2 numbers per site (C-A7)
    o2 = Oracle(6, 0.5, 1.0, 2, seed=9)                   # energy from Eq. 1 = E(0) + accepted Delta E (as P4), under heat bath
    o2.set_dynamics("heatbath")
    E0 = o2.energy()
    o2.sweep(5)
    assert (o2.energy() == E0 + o2.dE_accum()).all()
    o3 = Oracle(6, 0.5, 0.0, 1, seed=9)                   # T = 0: energy never rises; dE = 0 moves are coin flips
    o3.set_dynamics("heatbath")
    E = o3.energy()
    for _ in range(6):
        o3.sweep(1)
        E2 = o3.energy()
        assert (E2 <= E).all()
        E = E2


# ----------------------------------------------------------------------------------------
# P14  full-vector C_4 (Eq. 3 with r a lattice vector, reading C-S8v)
# ----------------------------------------------------------------------------------------
def _pack_replica_q(q):
    """spin words whose replica overlap field is q (+-1 array [N]) in every disorder lane: replica (a) all up,
    replica (b) = q."""
    hi = np.where(q < 0, np.uint64(0xFFFFFFFF00000000), np.uint64(0)).astype(np.uint64)
    return hi


def test_P14_vector_c4_against_the_3d_fft_and_its_symmetries():
    L, R = 6, 3
    o = Oracle(L, 0.5, 1.2, 2, seed=wl.seed_for(2, 5))
    o.sweep(4)
    S = unpack(o.get_spins())
    q3 = (S[:32] * S[32:]).reshape(32, L, L, L).astype(np.float64)         # [b][z][y][x]
    F = np.fft.fftn(q3, axes=(1, 2, 3))
    corr = np.rint(np.fft.ifftn(F * np.conj(F), axes=(1, 2, 3)).real).astype(np.int64)  # [b][dz][dy][dx] circular
    for dz in range(-R, R + 1):
        for dy in range(-R, R + 1):
            for dx in range(-R, R + 1):
                B = o.c4_vector(dx, dy, dz)
                assert (B == corr[:, dz % L, dy % L, dx % L]).all(), (dx, dy, dz)  # library routine (Wiener-Khinchin)
                assert (B == o.c4_vector(-dx, -dy, -dz)).all()                      # B(r) = B(-r)
    assert (o.c4_vector(0, 0, 0) == o.N).all()
    for d, e in enumerate(((1, 0, 0), (0, 1, 0), (0, 0, 1))):
        for r in range(R + 1):
            assert (o.c4_vector(r * e[0], r * e[1], r * e[2]) == o.c4_one(d, r)).all()  # the axis special case
    total = sum(o.c4_vector(dx, dy, dz) for dz in range(L) for dy in range(L) for dx in range(L))
    assert (total == o.overlap() ** 2).all()                               # sum over the torus = (sum_i q_i)^2


def test_P14_vector_c4_on_hand_made_overlap_fields():
    """Anisotropic fields whose correlation is known in closed form: a transposed or mis-signed displacement
    component, or a wrong wrap, changes the value."""
    L = 6
    N = L ** 3
    x, y, z = np.meshgrid(np.arange(L), np.arange(L), np.arange(L), indexing="ij")
    site = (x + L * (y + L * z)).ravel()
    o = Oracle(L, 0.5, 0.8, 2, seed=1)
    for name, field, expect in (
            ("stripes along x", (-1) ** x, lambda dx, dy, dz: N * (-1) ** dx),
            ("period-3 along y", np.where(y % 3 == 0, -1, 1), lambda dx, dy, dz: N if dy % 3 == 0 else -N // 3),
            ("planes z<2", np.where(z < 2, -1, 1), lambda dx, dy, dz: N - 4 * L * L * min(abs(dz) % L, L - abs(dz) % L, 2)),
    ):
        q = np.empty(N, dtype=np.int64)
        q[site] = np.asarray(field).ravel()
        o.set_spins(_pack_replica_q(q))
        for (dx, dy, dz) in ((1, 0, 0), (0, 1, 0), (0, 0, 1), (2, 1, 0), (-1, 2, 3), (3, -2, 1), (0, 3, -2), (1, 1, 1)):
            assert (o.c4_vector(dx, dy, dz) == expect(dx, dy, dz)).all(), (name, dx, dy, dz)
    q = np.ones(N, dtype=np.int64)
    q[4 + L * (1 + L * 3)] = -1                                                # one defect: two terms change sign
    o.set_spins(_pack_replica_q(q))
    assert (o.c4_vector(2, -1, 3) == N - 4).all() and (o.c4_vector(0, 0, 0) == N).all()


def test_P14_shell_sums_and_multiplicities():
    L, R = 8, 3
    o = Oracle(L, 0.6, 1.0, 2, seed=wl.seed_for(2, 6))
    o.sweep(3)
    S, mult = o.c4_shells(R)
    assert S.shape == (3 * R * R + 1, 32)
    count = {}
    for dz in range(-R, R + 1):
        for dy in range(-R, R + 1):
            for dx in range(-R, R + 1):
                count[dx * dx + dy * dy + dz * dz] = count.get(dx * dx + dy * dy + dz * dz, 0) + 1
    assert [int(m) for m in mult] == [count.get(d2, 0) for d2 in range(3 * R * R + 1)]
    assert [int(m) for m in mult[:7]] == [1, 6, 12, 8, 6, 24, 24]          # r^2 = 0..6: the cubic-lattice shells
    assert int(mult[7]) == 0 and (S[7] == 0).all()                         # 7 is not a sum of three squares
    assert (S[0] == o.N).all()
    B = o.c4(R)
    assert (S[1] == 2 * (B[0][1] + B[1][1] + B[2][1])).all()               # shell 1 = the six axis neighbours
    assert (S[3] == sum(o.c4_vector(a, b, c) for a in (-1, 1) for b in (-1, 1) for c in (-1, 1))).all()
    assert int(mult.sum()) == (2 * R + 1) ** 3
    full, _ = o.c4_shells(L // 2)                                          # +-L/2 are visited as two vectors
    assert (full[3 * (L // 2) ** 2] == 8 * o.c4_vector(L // 2, L // 2, L // 2)).all()


# ----------------------------------------------------------------------------------------
# P15  integral estimator of the coherence length (Eq. 5-6; reading C-S12)
# ----------------------------------------------------------------------------------------
def test_P15_c4_curve_is_mean_and_standard_error_over_the_disorder_samples():
    rng = np.random.default_rng(3)
    N, R = 512, 2
    mult = np.array([1, 6, 12, 8, 6, 24, 24, 0, 12, 30, 24, 24, 8], dtype=np.int64)
    S = rng.integers(-50, 400, size=(13, 32)) * mult[:, None]
    r, c, e = oracle.c4_curve(S, mult, N, R)
    d2s = [d2 for d2 in range(13) if mult[d2] and d2 <= R * R]
    assert np.allclose(r, np.sqrt(d2s), rtol=0, atol=1e-15)
    per = np.array([S[d2] / (mult[d2] * N) for d2 in d2s])
    assert np.allclose(c, per.mean(axis=1), rtol=1e-14)
    assert np.allclose(e, per.std(axis=1, ddof=1) / math.sqrt(32), rtol=1e-12)   # library routine


def test_P15_integral_estimator_closed_forms_and_cut_off():
    R = 8.0
    r = np.linspace(0.0, R, 9)
    c = 1.0 - r / R                                                        # linear: trapezoid is exact for k = 0
    I0, I1, xi, r_cut = oracle.integral_estimator(r, c, np.zeros_like(r), 0)
    assert abs(I0 - R / 2) < 1e-14 and r_cut == R
    assert abs(I1 - (R * R / 6 - 1.0 / 6)) < 1e-12                         # trapezoid of r(1 - r/R) with h = 1: exact - h^2 R/(6 R)... = R^2/6 - 1/6
    assert abs(xi - I1 / I0) < 1e-15
    xi0 = 2.5
    r = np.linspace(0.0, 60.0, 6001)                                       # fine grid: trapezoid -> the integral
    c = np.exp(-r / xi0)
    I1, I2, xi1, _ = oracle.integral_estimator(r, c, np.zeros_like(r), 1)
    assert abs(I1 - xi0 ** 2) < 1e-4 and abs(I2 - 2 * xi0 ** 3) < 1e-3 and abs(xi1 - 2 * xi0) < 1e-4  # int r^k e^{-r/xi} = k! xi^{k+1}
    assert np.isclose(I1, np.trapezoid(r * c, r), rtol=1e-12)              # library routine on the same grid
    e = np.full_like(r, 1e-3)                                              # 3 e = 3e-3 is crossed at r = xi0 ln(1/3e-3) = 14.52
    I1c, I2c, _, r_cut = oracle.integral_estimator(r, c, e, 1)
    j = int(np.argmax(c < 3e-3))
    assert r_cut == r[j - 1] and abs(r_cut - xi0 * math.log(1 / 3e-3)) < 0.02
    assert np.isclose(I1c, np.trapezoid((r * c)[:j], r[:j]), rtol=1e-12)
    assert np.isclose(I2c, np.trapezoid((r * r * c)[:j], r[:j]), rtol=1e-12)
    c2 = c.copy()
    c2[5] = -1.0                                                           # a dip below 3 e ends the integral there, even if C_4 recovers
    assert oracle.integral_estimator(r, c2, e, 1)[3] == r[4]


# ----------------------------------------------------------------------------------------
# P12  initial state
# ----------------------------------------------------------------------------------------
def test_P12_initial_state_statistics_and_replica_structure():
    L = 16
    N = L ** 3
    for p in (0.5, 0.77, 0.9):
        o = Oracle(L, p, 0.8, 2, seed=wl.seed_for(9))
        J = o.bond_bytes()
        assert (J[:32] == J[32:]).all()                                    # same bonds in both replicas (:33)
        n = 32 * 3 * N
        neg = int((J[:32] < 0).sum())
        assert abs(neg - n * (1 - p)) < 5 * math.sqrt(n * p * (1 - p))     # iid Bernoulli(1 - p) (:25)
        per_lane = (J[:32] < 0).reshape(32, -1).mean(axis=1)
        assert np.abs(per_lane - (1 - p)).max() < 6 * math.sqrt(p * (1 - p) / (3 * N))
        S = o.spin_bytes()
        assert abs(int((S < 0).sum()) - 32 * N) < 5 * math.sqrt(64 * N / 4)  # random start (:29)
        assert (S[:32] != S[32:]).any()                                    # replicas start differently (:33)
    a, b, c = Oracle(4, 0.5, 0.8, 1, seed=1), Oracle(4, 0.5, 0.8, 1, seed=1), Oracle(4, 0.5, 0.8, 1, seed=2)
    assert (a.get_spins() == b.get_spins()).all() and (a.get_bonds() == b.get_bonds()).all()
    assert (a.get_spins() != c.get_spins()).any() and (a.get_bonds() != c.get_bonds()).any()
    ind = Oracle(8, 0.5, 0.8, 1, seed=3).bond_bytes()
    assert (ind[:32] != ind[32:]).any()                                    # 64 independent samples


def test_create_rejects_bad_parameters():
    for args in ((3, 0.5, 0.8, 1), (0, 0.5, 0.8, 1), (4, 1.5, 0.8, 1), (4, 0.5, -1.0, 1), (4, 0.5, 0.8, 3),
                 (4, float("nan"), 0.8, 1), (4, 0.5, float("nan"), 1)):
        with pytest.raises(ValueError):
            Oracle(*args)
