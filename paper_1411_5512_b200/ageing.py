"""The paper's measurement protocol as a driver over the C ABI.

"Simulations start with random initial configurations ... We then examine the system at different waiting times t_w
(measured in sweeps) after the beginning of the simulation" (:29): at every t_w the configuration is kept (a device
snapshot; the paper wrote it to disk, :108) and C_4(r, t_w) (Eq. 3), q (Eq. 2), E and M are taken; afterwards, at
every t_w + t of the time grid, C(t, t_w) (Eq. 7) is taken against each snapshot that is old enough.

The library is grid-agnostic; the grids are the harness's: t_w = 10^k, t on the {1, 2, 5} x 10^m grid (S10).
Everything returned is the per-sample INTEGER sum (A = N C, B = N C_4, ...); averaging over samples and error bars
are the caller's (C-S9).  No arithmetic of the method happens here: this module only sequences ea_sweep /
ea_snapshot / ea_autocorr / ea_c4 / ea_energy / ea_magnetisation calls.
"""
import numpy as np


def decade_grid(t_max, mantissas=(1, 2, 5)):
    """1, 2, 5, 10, 20, 50, ... <= t_max."""
    out, m = [], 1
    while m <= t_max:
        out.extend(v * m for v in mantissas if v * m <= t_max)
        m *= 10
    return out


def run(sim, t_w_list, t_list, r_max=None, shells_r_max=None):
    """Advance `sim` (a binding.Sim at t = 0 with n_slots >= len(t_w_list)) through the protocol.

    Returns a dict:
      "t_w": [...], "t": [...],
      "A"[i][j]   int64 [64]   = sum_i S_i(t_w[i]) S_i(t_w[i] + t[j])            (Eq. 7), for every pair
      "B"[i]      int64 [3][r_max+1][32], "q"[i] int64 [32]  at t_w[i]           (Eq. 3, Eq. 2; 2-replica sims)
      "S"[i], "mult"[i]  shell sums of the full-vector C_4 at t_w[i] if shells_r_max is given
      "E"[i], "M"[i]     int64 [64] at t_w[i]                                   (Eq. 1; C-S14)
    """
    t_w_list = sorted(int(t) for t in t_w_list)
    t_list = sorted(int(t) for t in t_list)
    if len(t_w_list) > sim.n_slots:
        raise ValueError("the sim needs one snapshot slot per waiting time (%d > %d)" % (len(t_w_list), sim.n_slots))
    if sim.time != 0:
        raise ValueError("the protocol starts from the random start, t = 0 (PAPER.md:29)")
    events = {}  # absolute time -> list of ("snap", i) / ("corr", i, j)
    for i, tw in enumerate(t_w_list):
        events.setdefault(tw, []).append(("snap", i))
        for j, t in enumerate(t_list):
            events.setdefault(tw + t, []).append(("corr", i, j))
    res = {"t_w": t_w_list, "t": t_list, "A": [[None] * len(t_list) for _ in t_w_list], "E": [None] * len(t_w_list),
           "M": [None] * len(t_w_list)}
    two = sim.n_replicas == 2
    if two and r_max is not None:
        res["B"], res["q"] = [None] * len(t_w_list), [None] * len(t_w_list)
    if two and shells_r_max is not None:
        res["S"], res["mult"] = [None] * len(t_w_list), [None] * len(t_w_list)
    for when in sorted(events):
        sim.sweep(when - sim.time)
        for ev in sorted(events[when], key=lambda e: e[0] != "snap"):  # snapshots first: t = 0 pairs see them
            if ev[0] == "snap":
                i = ev[1]
                sim.snapshot(i)
                res["E"][i], res["M"][i] = sim.energy(), sim.magnetisation()
                if "B" in res:
                    res["B"][i], res["q"][i] = sim.c4(r_max, with_q=True)
                if "S" in res:
                    res["S"][i], res["mult"][i] = sim.c4_shells(shells_r_max)
            else:
                _, i, j = ev
                res["A"][i][j] = sim.autocorr(i)
    return res
