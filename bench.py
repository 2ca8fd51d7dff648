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
ea_get_spins (D2H), wall clock; `roofline` = the half-sweep kernel against the alu-pipe (LOP3) issue rate measured in the same run
(ea_selftest_pipes), with the HBM figure as a secondary record; `protocol` / `cfg5` = SURVEY 8(d)'s sweeps-only windows;
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

# Algorithmic alu-pipe work of one site word (64 attempts): 12 XOR (six bond x neighbour words per
# 32-sample half) + 8 full-adder LOP3 + 4 flip-rule LOP3 + 2 for the rare-level test + 9.5 Philox XOR3 + 8.5 Philox
# IMAD.WIDE (one block per two site words; an IMAD.WIDE takes an alu issue slot) = 44 slots, less the 2 of the two
# launch-uniform rounds that fold away = 42; addressing and the rare levels themselves are not counted.
ALGORITHMIC_ALU_INST_PER_SITE_WORD = 42
# fallback alu peak if ea_selftest_pipes fails: one warp instruction per 2 clocks per SM sub-partition (B300_MICROARCH
# "Pipe rates": rt_SMSP = 2) x 4 x 148 SMs at 1965 MHz
FALLBACK_ALU_WARP_INST_PER_S = 148 * 4 * 0.5 * 1.965e9


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
                    "snapshot + C(t,t_w) + C_4(r=0..L/2, 3 axes) + E + M (ea_snapshot + ea_measure)",
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
    pipes = None
    if rank == 0:  # the measured integer roofline, before the timed region
        try:
            pipes = binding.selftest_pipes(local_rank)
        except binding.EAError as e:
            sys.stderr.write("bench.py: ea_selftest_pipes failed (%s); using the guide's pipe rate\n" % e)

    def measure_point():
        sim.snapshot(0)
        rec = sim.measure(slot=0, r_max=r_max if cfg.n_replicas == 2 else None)  # ea_measure: A, B, q, E, M in one call
        return [rec[k] for k in ("A", "B", "q", "E", "M") if k in rec]

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
    from paper_1411_5512_b200 import census
    hbm_peak, hbm_src = measured_peak_gbs()
    t_half = t_sweeps / (2.0 * S * K)
    alg_bytes = algorithmic_bytes_per_half_sweep(N, cfg.n_replicas)
    kname = binding_kernel_name(sim.kernel)
    resident = kname == "resident" and S >= 8  # AUTO sends shorter calls through the ROWS launches
    hs_per_launch = 2 * S if resident else 1
    thr = [int(x) for x in sim.thresholds]
    variant = "always" if max(thr) >= 2 ** 32 else "rare" if thr[2] < 0x04000000 else "predicated"
    ckey = "resident_%s_%s" % ("u32" if cfg.n_replicas == 2 else "u64", variant) if resident else "k_sweep_%s" % kname
    cen, cen_note = census.lookup(ckey)
    if pipes is not None:
        alu_peak, alu_src = pipes["lop3_warp_inst_per_s"], "ea_selftest_pipes: dependent-free LOP3 stream on all SMs, measured in this run"
    else:
        alu_peak, alu_src = FALLBACK_ALU_WARP_INST_PER_S, "fallback: 148 SMs x 4 x 0.5 warp-inst/clk x 1.965 GHz (guide pipe rate)"
    alg_alu = ALGORITHMIC_ALU_INST_PER_SITE_WORD * (N // 2) / 32.0   # warp instructions per half-sweep
    roofline = {"bound": "alu", "kernel": "half-sweep (%s)" % ckey,
                "unit": "G warp-inst/s (alu pipe)", "peak": alu_peak / 1e9, "peak_source": alu_src,
                "achieved": None, "frac": None, "traffic": None,
                "half_sweeps_per_launch": hs_per_launch, "us_per_launch": 1e6 * t_half * hs_per_launch,
                "us_per_half_sweep": 1e6 * t_half, "share_of_step": t_sweeps / t_steps,
                "census": cen_note,
                "algorithmic": {"alu_warp_inst_per_half_sweep": alg_alu, "achieved": alg_alu / t_half / 1e9,
                                "frac": alg_alu / t_half / alu_peak,
                                "note": "%d alu-pipe instructions per site word is the method's own work (DESIGN.md 6); "
                                        "addressing, compares and moves are not counted" % ALGORITHMIC_ALU_INST_PER_SITE_WORD},
                "hbm": {"algorithmic_bytes_per_half_sweep": alg_bytes, "achieved_GBps": alg_bytes / t_half / 1e9,
                        "peak_GBps": hbm_peak, "peak_source": hbm_src,
                        "note": "secondary: inside a step the spins stay in shared memory and the bonds in L2, so the "
                                "algorithmic bytes do not cross HBM and this rate may exceed the HBM peak; see `traffic`"},
                "pipes_measured": pipes,
                "note": "achieved = alu-pipe issue slots per half-sweep = alu-pipe warp instructions + IMAD.WIDE (ncu counts of "
                        "THIS build, alu_census.json, refused if stale; an IMAD.WIDE takes an alu slot besides its fma-pipe "
                        "time: pipes_measured shows LOP3 at 4/5 of its rate with one IMAD.WIDE per four LOP3) / mean "
                        "half-sweep duration (CUDA events on the sim's stream around ea_sweep(S)); frac = achieved / "
                        "measured LOP3 issue rate of the whole chip"}
    if cen is not None:
        slots = cen.get("alu_slot_warp_inst_per_half_sweep", cen["alu_warp_inst_per_half_sweep"])
        alu_rate = slots / t_half
        roofline.update({"achieved": alu_rate / 1e9, "frac": alu_rate / alu_peak,
                         "alu_slot_warp_inst_per_half_sweep": slots,
                         "alu_warp_inst_per_half_sweep": cen["alu_warp_inst_per_half_sweep"],
                         "imad_wide_warp_inst_per_half_sweep": cen.get("imad_wide_warp_inst_per_half_sweep"),
                         "frac_alu_pipe_instructions_only": cen["alu_warp_inst_per_half_sweep"] / t_half / alu_peak,
                         "warp_inst_per_half_sweep": cen.get("warp_inst_per_half_sweep"),
                         "traffic": cen.get("dram_bytes_per_launch"),
                         "traffic_note": "dram bytes of the captured ncu launch (%g half-sweeps; cold L2): the lattice "
                                         "comes in once per launch" % cen.get("half_sweeps_in_captured_launch", 0),
                         "profile": cen.get("profile")})
    # ---- SURVEY 8(d) timing protocol: sweeps only, windows of n sweeps, 5 repeats, median and best -------------
    def sweep_window(sm, n, st):
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        with torch.cuda.stream(st):
            e0.record(st)
            sm.sweep(n)
            e1.record(st)
        e1.synchronize()
        sm.synchronize()
        return e0.elapsed_time(e1) * 1e-3

    protocol = None
    if args.protocol_window > 0:
        ts = sorted(sweep_window(sim, args.protocol_window, stream) for _ in range(5))
        per = lambda t: {"us_per_half_sweep": 1e6 * t / (2.0 * args.protocol_window),
                         "ps_per_attempt": 1e12 * t / (args.protocol_window * float(N) * LANES)}
        protocol = {"what": "SURVEY 8(d): CUDA events around ea_sweep(n), sweeps only, 5 repeats", "config": cfg.name,
                    "n_sweeps": args.protocol_window, "median": per(ts[2]), "best": per(ts[0]), "worst": per(ts[4])}
    # ---- cfg5: one window per (p, T) point of the paper's production family ------------------
    cfg5 = None
    if args.cfg5_window > 0 and ws == 1:
        pts = []
        for name in sorted(k for k in wl.CONFIGS if k.startswith("cfg5_")):
            c5 = wl.CONFIGS[name]
            s5 = binding.Sim(c5.L, c5.p, c5.T, n_replicas=c5.n_replicas, seed=c5.seed, n_slots=0, kernel=args.kernel,
                             device=local_rank, stream=stream)
            s5.sweep(100)  # warm-up 100 sweeps
            s5.synchronize()
            t5 = sweep_window(s5, args.cfg5_window, stream)
            pts.append({"config": name, "p": c5.p, "T": c5.T, "kernel": binding_kernel_name(s5.kernel),
                        "us_per_half_sweep": 1e6 * t5 / (2.0 * args.cfg5_window),
                        "ps_per_attempt": 1e12 * t5 / (args.cfg5_window * float(c5.N) * LANES)})
            s5.close()
        by_T = {}
        for q in pts:
            by_T.setdefault(q["T"], []).append(q["us_per_half_sweep"])
        cfg5 = {"what": "one %d-sweep window per (p, T) point of BASELINE.json configs[4], sweeps only, after 100 warm-up "
                        "sweeps (the paper ran 10^8 sweeps per point, PAPER.md:108)" % args.cfg5_window,
                "n_sweeps": args.cfg5_window, "points": pts,
                "spread_in_p": {str(T): (max(v) - min(v)) / min(v) for T, v in by_T.items()}}
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

    if next_rows is not None and ws == 1:
        # single small lattices (BASELINE configs[0..1] and the paper's scans at L = 32): SMALL keeps spins and
        # bonds in the shared memory of one CTA / one thread-block cluster for the whole ea_sweep call
        small = []
        for name, Ls, n_rep, n_sm in (("cfg1", 8, 1, 20000), ("L16", 16, 2, 20000), ("cfg2", 32, 2, 20000)):
            ss = binding.Sim(Ls, 0.5, cfg.T, n_replicas=n_rep, seed=seed + 2000 + Ls, n_slots=0, device=local_rank, stream=stream)
            ss.sweep(100)
            ss.synchronize()
            t_s = sweep_window(ss, n_sm, stream)
            small.append({"config": name, "L": Ls, "n_replicas": n_rep, "kernel": binding_kernel_name(ss.kernel),
                          "us_per_half_sweep": 1e6 * t_s / (2.0 * n_sm), "ps_per_attempt": 1e12 * t_s / (n_sm * float(Ls) ** 3 * LANES)})
            ss.close()
        next_rows["small_lattices"] = {"what": "one sim alone, CUDA events around ea_sweep(20000) after 100 warm-up sweeps", "points": small}

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
        "protocol": protocol,
        "cfg5": cfg5,
        "next_rows": next_rows,
        "wall_s_timed_loop": wall,
        "paper_context": "paper: ~8 ps per spin flip on a GeForce GTX 570 (PAPER.md:5, :92) -- other hardware, "
                         "context only",
    }
    print(json.dumps(line))
    return 0


def binding_kernel_name(k):
    return {1: "scalar", 2: "vec2", 3: "rows", 4: "resident", 5: "fold", 6: "rows_persistent", 7: "small"}.get(int(k), str(k))


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
    ap.add_argument("--protocol-window", type=int, default=10000,
                    help="sweeps per window of the SURVEY 8(d) protocol (5 repeats, median / best); 0 = skip")
    ap.add_argument("--cfg5-window", type=int, default=100000,
                    help="sweeps per (p, T) point of the cfg5 family (SURVEY 8(d) asks for up to 10^6); 0 = skip")
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
