#!/usr/bin/env python
"""bench.py -- ps per spin-flip attempt of the checkerboard Metropolis hot path on B200.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--impl ours|reference]
                    [--config cfg4] [--sweeps-per-step S] [--kernel auto]

A STEP is one pass of the whole hot path over one batch of 64 samples: S full
sweeps (a1-a7: 2 S half-sweeps; at L = 128 one persistent RESIDENT launch) followed by one measure point -- snapshot (a8), C(t,t_w) (a9),
overlap + C_4(r) for r = 0..L/2 on the three axes (a10), energy (a11), magnetisation (a12).  The lattice
(setup, a0) is drawn once on the device before the timed region.  In the paper's workload the measure
points are log-spaced, i.e. far rarer than one per S = 1000 sweeps, so this over-weights the
observables.

Workload: BASELINE.json configs[3] (cfg4): L = 128, p = 0.77, T = 0.8, 32 disorders x 2 replicas -- the
L = 128 configuration the metric and its 70 % target are quoted on.  All inputs are seeded and synthetic,
which is what the paper's inputs are (random +-J bonds, random start).

The JSON line: `value` = device-timed ps per attempt with the lattice resident in HBM; `e2e` = the same
through the C ABI with HOST buffers (pinned): ea_set_bonds + ea_set_spins (H2D) -> sweeps -> observables ->
ea_get_spins (D2H), wall clock; `roofline` = the half-sweep kernel against the measured HBM copy bandwidth;
`cpu_baseline` = the CPU oracle on this box's host cores on a bounded sample.

N > 1 (torchrun): replicas only -- every rank runs its own independent batch (seed + rank); no collective
on the data path; time = max over ranks; value = whole-job ps per attempt.
"""
import argparse
import json
import os
import subprocess
import sys
import threading
import time

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

import numpy as np  # noqa: E402

from paper_1411_5512_b200 import replicas  # noqa: E402
from paper_1411_5512_b200 import workloads as wl  # noqa: E402

METRIC = "ps per spin-flip attempt"
UNIT = "ps/attempt"
LANES = 64
FALLBACK_HBM_GBS = 6650.0  # /opt/skills/guides/B200_PROFILING.md, used only if MEASURED_PEAKS.json is absent

# From the `ncu --set full` captures summarised in profiles/ (each .md names its command), per kernel variant:
#   traffic  = dram__bytes_read.sum + dram__bytes_write.sum of ONE launch at the bench configuration (cold L2: ncu
#              flushes the caches before the launch).  ROWS: one launch = one half-sweep.  RESIDENT: one launch =
#              the whole ea_sweep(S) call (2 S half-sweeps): the lattice is read once and written back once.
#   alu_inst = sm__inst_executed_pipe_alu.sum per half-sweep (warp instructions on the LOP3/ISETP pipe).
NCU = {
    "rows": {"traffic": 41996032, "alu_inst": None, "profile": "profiles/r01_ncu_full_k_sweep_rows.md"},
    "resident": {"traffic": 42000000 + 255000, "alu_inst": 631011472 / 400.0,  # profiles/r01_launches_resident.md
                 "profile": "profiles/r01_ncu_full_k_sweep_resident.md"},
}
# alu pipe: one warp instruction per 2 clocks per SM sub-partition (B300_MICROARCH "Pipe rates": rt_SMSP = 2),
# 4 sub-partitions x 148 SMs, at the max SM clock of MEASURED_PEAKS.json (1965 MHz): DESIGN.md section 6
ALU_PEAK_WARP_INST_PER_S = 148 * 4 * 0.5 * 1.965e9


def algorithmic_bytes_per_half_sweep(N, n_replicas):
    """spins read N/2 (own) + N/2 (neighbours) + written N/2 words of 8 B = 12 N bytes;
    bonds: each of the 3 N bonds touches exactly one updated site -> 3 N words of 4 B (2 replicas share the
    32 disorder bits) or 8 B (64 independent samples)."""
    return 12 * N + 3 * N * (4 if n_replicas == 2 else 8)


def measured_peak_gbs():
    path = os.path.join(ROOT, "MEASURED_PEAKS.json")
    try:
        with open(path) as f:
            return float(json.load(f)["hbm_gbs"]), "MEASURED_PEAKS.json hbm_gbs (measured)"
    except Exception:
        return FALLBACK_HBM_GBS, "fallback (B200_PROFILING.md)"


class ClockSampler:
    """nvidia-smi clocks / throttle reasons DURING the timed region (B200_PROFILING.md, the clocks line)."""
    Q = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,"
         "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,"
         "clocks_event_reasons.sw_power_cap")
    NAMES = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]

    def __init__(self, index):
        self.index, self.rows, self.proc, self.thread = index, [], None, None
        self._nvml_stop, self._nvml_rows = None, None

    def _nvml_loop(self, pynvml, handle):
        """The same quantities straight from NVML every ~5 ms: the timed region of the default run lasts 0.1 s, which a
        100 ms nvidia-smi loop samples once."""
        bits = [("hw_slowdown", pynvml.nvmlClocksThrottleReasonHwSlowdown),
                ("hw_thermal_slowdown", pynvml.nvmlClocksThrottleReasonHwThermalSlowdown),
                ("sw_thermal_slowdown", pynvml.nvmlClocksThrottleReasonSwThermalSlowdown),
                ("sw_power_cap", pynvml.nvmlClocksThrottleReasonSwPowerCap)]
        mx = pynvml.nvmlDeviceGetMaxClockInfo(handle, pynvml.NVML_CLOCK_SM)
        while not self._nvml_stop.is_set():
            try:
                sm = pynvml.nvmlDeviceGetClockInfo(handle, pynvml.NVML_CLOCK_SM)
                pw = pynvml.nvmlDeviceGetPowerUsage(handle) / 1000.0
                rs = pynvml.nvmlDeviceGetCurrentClocksThrottleReasons(handle)
                self._nvml_rows.append((float(sm), float(mx), pw, [n for n, b in bits if rs & b]))
            except Exception:
                pass
            time.sleep(0.005)

    def start(self):
        try:  # NVML first (fast), nvidia-smi as the fallback
            import pynvml
            pynvml.nvmlInit()
            handle = pynvml.nvmlDeviceGetHandleByIndex(self._physical_index())
            self._nvml_stop, self._nvml_rows = threading.Event(), []
            self.thread = threading.Thread(target=self._nvml_loop, args=(pynvml, handle), daemon=True)
            self.thread.start()
            return
        except Exception:
            self._nvml_stop, self._nvml_rows = None, None
        try:
            self.proc = subprocess.Popen(["nvidia-smi", "-i", str(self.index), "--query-gpu=" + self.Q,
                                          "--format=csv,noheader,nounits", "-lms", "100"],
                                         stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
        except OSError:
            self.proc = None
            return
        self.thread = threading.Thread(target=self._read, daemon=True)
        self.thread.start()

    def _read(self):
        for line in self.proc.stdout:
            self.rows.append([x.strip() for x in line.split(",")])

    def _physical_index(self):
        vis = os.environ.get("CUDA_VISIBLE_DEVICES")
        if vis:
            try:
                return int(vis.split(",")[self.index])
            except (ValueError, IndexError):
                pass
        return self.index

    def stop(self):
        if self._nvml_stop is not None:
            self._nvml_stop.set()
            self.thread.join(timeout=2)
            rows = self._nvml_rows
            reasons = sorted({r for row in rows for r in row[3]})
            return {"sm_mhz": float(np.median([r[0] for r in rows])) if rows else None,
                    "sm_max_mhz": max(r[1] for r in rows) if rows else None,
                    "power_w_max": max(r[2] for r in rows) if rows else None, "reasons": reasons, "samples": len(rows),
                    "source": "nvml, every 5 ms during the timed region"}
        if self.proc is None:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": [], "samples": 0}
        self.proc.terminate()
        try:
            self.proc.wait(timeout=5)
        except Exception:
            self.proc.kill()
        self.thread.join(timeout=5)
        sm, mx, pw, reasons = [], [], [], set()
        for r in self.rows:
            try:
                sm.append(float(r[0])); mx.append(float(r[1])); pw.append(float(r[2]))
            except (ValueError, IndexError):
                continue
            for name, v in zip(self.NAMES, r[3:7]):
                if v.lower().startswith("active"):
                    reasons.add(name)
        return {"sm_mhz": float(np.median(sm)) if sm else None, "sm_max_mhz": max(mx) if mx else None,
                "power_w_max": max(pw) if pw else None, "reasons": sorted(reasons), "samples": len(sm)}


# ----------------------------------------------------------------------------------------------------------
# the CPU oracle, timed as it stands (cpu_baseline leg and --impl reference).  The ONLY place bench.py
# touches oracle/.
# ----------------------------------------------------------------------------------------------------------
def time_oracle(cfg, S, steps, warmup):
    """Times the oracle on a bounded sample of the step: `steps` x (1 sweep) after `warmup` x (1 sweep), plus
    ONE measure point (snapshot, C, C_4 r=0..L/2, E, M).  ps/attempt is that of a whole step, extrapolated:
    (S * t_sweep + t_observables) / (S * N * 64)."""
    import oracle
    o = oracle.Oracle(cfg.L, cfg.p, cfg.T, n_replicas=cfg.n_replicas, seed=cfg.seed, n_slots=1)
    cores = oracle.max_threads()
    for _ in range(warmup):
        o.sweep(1)
    per = []
    for _ in range(steps):
        t0 = time.perf_counter()
        o.sweep(1)
        per.append(time.perf_counter() - t0)
    t_sweep = float(np.mean(per))
    # also one thread (the lanes are run one after the other), two sweeps
    t_one = None
    if hasattr(oracle, "set_threads"):
        oracle.set_threads(1)
        t0 = time.perf_counter()
        o.sweep(2)
        t_one = (time.perf_counter() - t0) / 2
        oracle.set_threads(cores)
    # one measure point; C_4 on bytes is the slow part (3 (L/2+1) passes over 32 N bytes), so it is timed on a
    # bounded sample -- r = 1 on each of the 3 axes -- and scaled by (L/2 + 1) (every r costs the same loop)
    t0 = time.perf_counter()
    o.snapshot(0)
    o.autocorr(0)
    o.energy()
    o.magnetisation()
    t_obs = time.perf_counter() - t0
    c4_note = "no C_4 (1 replica)"
    if cfg.n_replicas == 2:
        t0 = time.perf_counter()
        o.overlap()
        for d in range(3):
            o.c4_one(d, 1)
        t_c4 = time.perf_counter() - t0
        t_obs += t_c4 * (cfg.L // 2 + 1)
        c4_note = "C_4 timed at r=1 on 3 axes (%.3f s) x (L/2+1)=%d" % (t_c4, cfg.L // 2 + 1)
    o.close()
    step_s = S * t_sweep + (t_obs or 0.0)
    ps = 1e12 * step_s / (S * cfg.N * LANES)
    sample = ("oracle/ea_oracle.c as it stands (byte per spin, scalar Metropolis, OpenMP over the 64 samples): "
              "%d timed single sweeps of %s (L=%d) after %d warm-up sweeps, mean %.3f s/sweep; one measure point "
              "(snapshot, C, E, M; %s) %.3f s; value = (S*t_sweep + t_obs)/(S*N*64) at S=%d"
              % (steps, cfg.name, cfg.L, warmup, t_sweep, c4_note, t_obs, S))
    out = {"value": ps, "unit": UNIT, "cores": cores, "kind": "oracle", "sample": sample,
           "s_per_sweep": t_sweep, "s_per_measure_point": t_obs}
    if t_one is not None:
        out["one_thread"] = {"s_per_sweep": t_one, "ps_per_attempt_sweeps_only": 1e12 * t_one / (cfg.N * LANES)}
    return out, step_s


def run_reference(args, cfg):
    rank, _, ws = replicas.world()
    if rank != 0:
        return 0  # the oracle is one host program: rank 0 alone runs and prints it
    base, step_s = time_oracle(cfg, args.sweeps_per_step, args.steps, args.warmup)
    line = {
        "impl": "reference", "metric": METRIC, "value": base["value"], "unit": UNIT, "n_gpus": args.gpus,
        "steps": args.steps, "warmup": args.warmup, "ms_per_step": 1e3 * step_s, "higher_is_better": False,
        "scaling": "weak", "vs_baseline": None, "dtype": "int8", "data": "synthetic",
        "config": workload_config(cfg, args, ws),
        "cpu_baseline": {k: base[k] for k in ("value", "unit", "cores", "kind", "sample")},
        "e2e": {"value": base["value"], "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0,
    }
    print(json.dumps(line))
    return 0


def workload_config(cfg, args, ws):
    return {"workload": "BASELINE.json configs[%d] (%s): L=%d periodic 3D +-J EA, p=%g, T=%g, 64 samples = "
                        "%s in uint64 words"
                        % (int(cfg.name[3]) - 1, cfg.name, cfg.L, cfg.p, cfg.T,
                           "32 disorders x 2 replicas" if cfg.n_replicas == 2 else "64 independent"),
            "L": cfg.L, "N": cfg.N, "p": cfg.p, "T": cfg.T, "n_replicas": cfg.n_replicas,
            "sweeps_per_step": args.sweeps_per_step,
            "step": "S sweeps = 2S half-sweeps (RESIDENT at L=128: one persistent launch; else one launch per colour) + "
                    "snapshot + C(t,t_w) + C_4(r=0..L/2, 3 axes) + E + M",
            "l2": "flushed between timed steps (a %d MiB buffer is overwritten); inside a step the %.0f MiB "
                  "lattice is re-swept S times and stays on the chip (spins in shared memory, bonds in L2 for the "
                  "RESIDENT kernel; all of it in L2 for the per-colour kernels), as in the paper's 10^7-sweep runs"
                  % (args.flush_mib, (8 * cfg.N + 3 * cfg.N * (4 if cfg.n_replicas == 2 else 8)) / 2 ** 20),
            "parallelism": "replicas only: %d independent batch(es), one per GPU, no data-path collective" % ws}


# ----------------------------------------------------------------------------------------------------------
def run_ours(args, cfg):
    import torch
    from paper_1411_5512_b200 import binding

    rank, local_rank, ws = replicas.init()
    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device (there is no CPU fallback; use --impl reference for the oracle)")
    torch.cuda.set_device(local_rank)
    dev = torch.device("cuda", local_rank)
    stream = torch.cuda.Stream(device=dev)
    L, N, S, K, W = cfg.L, cfg.N, args.sweeps_per_step, args.steps, args.warmup
    seed = replicas.replica_seed(cfg.seed, rank)
    sim = binding.Sim(L, cfg.p, cfg.T, n_replicas=cfg.n_replicas, seed=seed, n_slots=1, kernel=args.kernel,
                      device=local_rank, stream=stream)
    flush = torch.empty(args.flush_mib << 20, dtype=torch.uint8, device=dev)
    r_max = L // 2

    def measure_point():
        sim.snapshot(0)
        out = [sim.autocorr(0)]
        if cfg.n_replicas == 2:
            out.append(sim.c4(r_max, with_q=True))
        out.append(sim.energy())
        out.append(sim.magnetisation())
        return out

    def step(timed):
        with torch.cuda.stream(stream):
            flush.zero_()  # L2 flush between steps, outside the timed events
            e0 = torch.cuda.Event(enable_timing=True)
            e1 = torch.cuda.Event(enable_timing=True)
            e2 = torch.cuda.Event(enable_timing=True)
            e0.record(stream)
            sim.sweep(S)
            e1.record(stream)
            obs = measure_point()
            e2.record(stream)
        if timed is not None:
            timed.append((e0, e1, e2))
        return obs

    for _ in range(W):
        step(None)
    torch.cuda.synchronize()
    replicas.barrier()
    clocks = ClockSampler(local_rank)
    if rank == 0:
        clocks.start()
    launches0 = sim.launch_count
    events = []
    torch.cuda.synchronize()
    wall0 = time.perf_counter()
    for _ in range(K):
        step(events)
    torch.cuda.synchronize()
    wall = time.perf_counter() - wall0
    replicas.barrier()
    launches = sim.launch_count - launches0
    clk = clocks.stop() if rank == 0 else None
    t_sweeps = sum(a.elapsed_time(b) for a, b, _ in events) * 1e-3
    t_steps = sum(a.elapsed_time(c) for a, _, c in events) * 1e-3
    t_max = replicas.max_over_ranks(t_steps)
    attempts_rank = float(K) * S * N * LANES
    attempts = replicas.sum_over_ranks(attempts_rank)
    value = 1e12 * t_max / attempts

    # ---- end to end through the C ABI with host buffers (pinned), wall clock --------------------------------
    h_spins = torch.empty(N, dtype=torch.int64).pin_memory()
    h_bonds = torch.empty(3 * N, dtype=torch.int64).pin_memory()
    h_out = torch.empty(N, dtype=torch.int64).pin_memory()
    sim.get_spins(out=h_spins)
    sim.get_bonds(out=h_bonds)
    obs_bytes = 0

    def e2e_step():
        sim.set_bonds(h_bonds)   # H2D 3N words (canonical 64-bit bond words)
        sim.set_spins(h_spins)   # H2D N words
        sim.sweep(S)
        obs = measure_point()
        sim.get_spins(out=h_out)  # D2H N words ("whole system configurations were ... stored")
        return obs

    for _ in range(max(1, min(W, 3))):
        obs = e2e_step()
    obs_bytes = sum(int(np.asarray(x).nbytes) if not isinstance(x, tuple) else sum(int(y.nbytes) for y in x)
                    for x in obs)
    torch.cuda.synchronize()
    replicas.barrier()
    k_e2e = max(1, min(K, 5))
    w0 = time.perf_counter()
    for _ in range(k_e2e):
        e2e_step()
    torch.cuda.synchronize()
    t_e2e = replicas.max_over_ranks(time.perf_counter() - w0)
    e2e_value = 1e12 * t_e2e / (replicas.sum_over_ranks(float(k_e2e) * S * N * LANES))

    if rank != 0:
        sim.close()
        return 0

    # ---- roofline of the dominant kernel (the half-sweep), measured live above ------------------------------
    peak, peak_src = measured_peak_gbs()
    t_half = t_sweeps / (2.0 * S * K)
    alg = algorithmic_bytes_per_half_sweep(N, cfg.n_replicas)
    achieved = alg / t_half / 1e9
    kname = binding_kernel_name(sim.kernel)
    resident = kname == "resident" and S >= 8  # AUTO sends shorter calls through the ROWS launches
    hs_per_launch = 2 * S if resident else 1
    ncu = NCU.get(kname, {})
    roofline = {"bound": "hbm", "kernel": "half-sweep (%s)" % kname,
                "achieved": achieved, "peak": peak, "unit": "GB/s", "frac": achieved / peak,
                "traffic": ncu.get("traffic"), "half_sweeps_per_launch": hs_per_launch,
                "algorithmic_bytes_per_launch": alg * hs_per_launch,
                "us_per_launch": 1e6 * t_half * hs_per_launch, "us_per_half_sweep": 1e6 * t_half,
                "peak_source": peak_src, "share_of_step": t_sweeps / t_steps, "profile": ncu.get("profile"),
                "note": "achieved = algorithmic bytes per launch / mean launch duration (CUDA events on the sim's "
                        "stream around ea_sweep(S)). north_star: the roofline is the slower of bytes / HBM bandwidth "
                        "and integer ops / issue rate -- HBM (7.7 us per half-sweep) is the slower one, so bound = "
                        "hbm; the lattice is L2-resident (ROWS) or shared-memory-resident (RESIDENT) inside a step, "
                        "so frac exceeds 1 and the alu figure below is the bound that then applies (DESIGN.md 6)"}
    if ncu.get("alu_inst"):
        alu_rate = ncu["alu_inst"] / t_half
        roofline["alu"] = {"achieved": alu_rate / 1e9, "peak": ALU_PEAK_WARP_INST_PER_S / 1e9,
                           "unit": "G warp-inst/s (alu pipe)", "frac": alu_rate / ALU_PEAK_WARP_INST_PER_S,
                           "alu_warp_inst_per_half_sweep": ncu["alu_inst"]}
    # ---- SURVEY 8(f) rows built so far, timed on the same state (not part of `value`) -----------------------
    next_rows = None
    if cfg.n_replicas == 2 and not args.no_next_rows:
        R = 8
        sim.c4_shells(2)  # warm-up (first-call allocations)
        torch.cuda.synchronize()
        w0 = time.perf_counter()
        S_sh, mult = sim.c4_shells(R)
        t_shells = time.perf_counter() - w0
        r_c, c_c, e_c = binding.c4_curve(S_sh, mult, N, R)
        xi = binding.integral_estimator(r_c, c_c, e_c, 1)
        n_vec = ((2 * R + 1) ** 3 - 1) // 2
        next_rows = {"c4_shells": {"r_max": R, "vectors_visited": n_vec, "ms": 1e3 * t_shells,
                                   "popc_lane_ops_per_s": n_vec * float(N) / t_shells,
                                   "popc_peak_per_s": 148 * 16 * 1.965e9,
                                   "note": "NEXT-1: ea_c4_shells wall time incl. transposition, job upload and D2H; "
                                           "bound = POPC rate (16 lanes/clk/SM); kernel alone: profiles/"},
                     "xi_1": {"I_1": xi[0], "I_2": xi[1], "xi_1": xi[2], "r_cut": xi[3], "t_w": int(sim.time)}}
    sim.close()
    if next_rows is not None and ws == 1:
        from paper_1411_5512_b200.scan import Scan
        Ls, Ks, n_sc = 64, 8, 2000
        sc = Scan([{"L": Ls, "p": 0.6 + 0.01 * k, "T": cfg.T, "seed": seed + 1000 + k} for k in range(Ks)], device=local_rank)
        sc.sweep(64)
        sc.synchronize()
        w0 = time.perf_counter()
        sc.sweep(n_sc)
        sc.synchronize()
        t_sc = time.perf_counter() - w0
        sc.close()
        next_rows["scan"] = {"L": Ls, "sims": Ks, "sweeps": n_sc, "ps_per_attempt_aggregate": 1e12 * t_sc / (Ks * n_sc * Ls ** 3 * 64.0),
                             "note": "NEXT-4 driver: K independent L=64 sims, one stream + CUDA graph each, issued back to back"}

    cpu_baseline = None
    if ws == 1 and not args.no_cpu_baseline:
        base, _ = time_oracle(cfg, S, steps=args.cpu_sweeps, warmup=1)
        cpu_baseline = {k: base[k] for k in ("value", "unit", "cores", "kind", "sample", "one_thread") if k in base}

    line = {
        "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": ws, "steps": K, "warmup": W,
        "ms_per_step": 1e3 * t_max / K, "higher_is_better": False, "scaling": "weak", "vs_baseline": None,
        "dtype": "u64", "data": "synthetic", "config": workload_config(cfg, args, ws),
        "clocks": clk,
        "e2e": {"value": e2e_value, "unit": UNIT, "h2d_bytes_per_step": 8 * 4 * N,
                "d2h_bytes_per_step": 8 * N + obs_bytes, "steps": k_e2e,
                "path": "ea_set_bonds + ea_set_spins (pinned host) -> ea_sweep(S) -> measure point -> ea_get_spins"},
        "gpu_launches": int(launches),
        "roofline": roofline,
        "cpu_baseline": cpu_baseline,
        "next_rows": next_rows,
        "wall_s_timed_loop": wall,
        "paper_context": "paper: ~8 ps per spin flip on a GeForce GTX 570 (PAPER.md:5, :92) -- other hardware, "
                         "context only",
    }
    print(json.dumps(line))
    return 0


def binding_kernel_name(k):
    return {1: "scalar", 2: "vec2", 3: "rows", 4: "resident"}.get(int(k), str(k))


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=10)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--config", default=wl.BENCH_CONFIG, choices=sorted(wl.CONFIGS))
    ap.add_argument("--sweeps-per-step", type=int, default=1000)
    ap.add_argument("--kernel", default="auto")
    ap.add_argument("--no-next-rows", action="store_true", help="skip the timing of the SURVEY 8(f) rows (c4_shells, scan)")
    ap.add_argument("--flush-mib", type=int, default=256)
    ap.add_argument("--cpu-sweeps", type=int, default=12, help="oracle sweeps timed for cpu_baseline")
    ap.add_argument("--no-cpu-baseline", action="store_true", help="skip the oracle timing (profiler runs)")
    args = ap.parse_args()
    if args.warmup < 3 and args.impl == "ours":
        args.warmup = 3  # timing rule: W >= 3
    cfg = wl.CONFIGS[args.config]
    if args.impl == "reference":
        return run_reference(args, cfg)
    return run_ours(args, cfg)


if __name__ == "__main__":
    sys.exit(main())
