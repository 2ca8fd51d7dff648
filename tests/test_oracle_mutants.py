"""Mutation check of the oracle's pins: every hand-made mutant of oracle/ea_oracle.c -- a plausible
mistake in one line -- must make the pin named beside it fail, and the unmodified source must pass the same pins.

Each mutant is built into a temporary library (gcc, as oracle/build.py does) and the pin tests run against it in a
subprocess (EA_ORACLE_LIB points the oracle loader at it).  CPU only.
"""
import os
import subprocess
import sys
import tempfile
from concurrent.futures import ThreadPoolExecutor

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
SRC = os.path.join(ROOT, "oracle", "ea_oracle.c")

# (name, text in the source (exactly one occurrence), replacement, pin expected to fail)
MUTANTS = [
    ("exponent factor 2 instead of 4 (Eq. 9 with the 2/T and the factor 2 of Delta E)",
     "double prob = exp(-(4.0 * (double)(3 - n_u)) / T);", "double prob = exp(-(2.0 * (double)(3 - n_u)) / T);",
     "test_P3_thresholds_golden_and_closed_form"),
    ("threshold truncated instead of rounded",
     "thr[n_u] = (uint64_t)floor(4294967296.0 * prob + 0.5);\n    }\n}\n\n/* Heat-bath variant",
     "thr[n_u] = (uint64_t)floor(4294967296.0 * prob);\n    }\n}\n\n/* Heat-bath variant",
     "test_P3_thresholds_golden_and_closed_form"),
    ("'<=' for '<' in the Metropolis decision",
     "/* 0, 1 or 2 */\n    return (uint64_t)r < thr[n_u];", "/* 0, 1 or 2 */\n    return (uint64_t)r <= thr[n_u];",
     "test_P3_single_spin_decision_at_the_threshold_edges"),
    ("Delta E = 0 rejected",
     "if (local_sum <= 0) return 1;", "if (local_sum < 0) return 1;\n    if (local_sum == 0) return 0;",
     "test_P3_single_spin_decision_at_the_threshold_edges"),
    ("wrong neighbour: -y bond multiplied by the +y spin",
     "sum += J[1 * N + ym] * S[site] * S[ym];", "sum += J[1 * N + ym] * S[site] * S[yp];",
     "test_P4_energy_from_eq1_equals_accumulated_delta_e"),
    ("wrong bond owner: own +x bond used for the -x neighbour",
     "sum += J[0 * N + xm] * S[site] * S[xm];", "sum += J[0 * N + site] * S[site] * S[xm];",
     "test_P7_gauge_transformation_commutes_with_the_dynamics"),
    ("replica halves swap their random numbers",
     "uint32_t r = lane < 32 ? s->r_lo[site] : s->r_hi[site];", "uint32_t r = lane < 32 ? s->r_hi[site] : s->r_lo[site];",
     "test_stream_layout_of_update_numbers"),
    ("colour tags swapped in the counter",
     "uint32_t tag = parity == 0 ? TAG_UPDATE_PARITY0 : TAG_UPDATE_PARITY1;",
     "uint32_t tag = parity == 0 ? TAG_UPDATE_PARITY1 : TAG_UPDATE_PARITY0;",
     "test_stream_layout_of_update_numbers"),
    ("second site of a pair takes the words of the first",
     "s->r_lo[site] = out[2 * second];", "s->r_lo[site] = out[second];",
     "test_stream_layout_of_update_numbers"),
    ("colour order of a sweep swapped",
     "oracle_half_sweep(s, 0);\n        oracle_half_sweep(s, 1);", "oracle_half_sweep(s, 1);\n        oracle_half_sweep(s, 0);",
     "test_P2_oracle_one_sweep_transitions_match_the_exact_boltzmann_metropolis_matrix"),
    ("energy over backward instead of forward bonds",
     "S[oracle_neighbour(s->L, site, d, +1)];", "S[oracle_neighbour(s->L, site, d, -1)];",
     "test_P4_energy_from_eq1_equals_accumulated_delta_e"),
    ("C_4 along the wrong axis",
     "int64_t other = oracle_shift(s->L, site, d, r); /* i + r e_d */", "int64_t other = oracle_shift(s->L, site, (d + 1) % 3, r);",
     "test_P11_observables_against_numpy_and_fft"),
]


def build(source_text, out_dir, tag):
    c_path = os.path.join(out_dir, "ea_oracle_%s.c" % tag)
    lib = os.path.join(out_dir, "libea_oracle_%s.so" % tag)
    with open(c_path, "w") as f:
        f.write(source_text)
    subprocess.run(["gcc", "-std=c99", "-O2", "-fopenmp", "-fPIC", "-shared", "-o", lib, c_path, "-lm"], check=True)
    return lib


def run_pins(lib, names):
    env = dict(os.environ, EA_ORACLE_LIB=lib, OMP_NUM_THREADS="2")
    k = " or ".join(sorted(set(names)))
    return subprocess.run([sys.executable, "-m", "pytest", os.path.join(ROOT, "tests", "test_oracle_pins.py"), "-x", "-q",
                           "-p", "no:cacheprovider", "-k", k], env=env, cwd=ROOT, capture_output=True, text=True)


def test_every_mutant_of_the_oracle_fails_its_pin_and_the_original_passes():
    with open(SRC) as f:
        src = f.read()
    with tempfile.TemporaryDirectory() as tmp:
        jobs = []
        for i, (name, old, new, pin) in enumerate(MUTANTS):
            assert src.count(old) == 1, "mutant %r: its source line was not found exactly once (oracle changed?)" % name
            jobs.append((name, build(src.replace(old, new), tmp, "m%d" % i), [pin]))
        control = build(src, tmp, "control")
        with ThreadPoolExecutor(max_workers=4) as ex:
            results = list(ex.map(lambda j: run_pins(j[1], j[2]), jobs))
            ok = run_pins(control, [m[3] for m in MUTANTS])
        assert ok.returncode == 0, "the unmodified oracle fails its pins in this harness:\n" + ok.stdout[-2000:]
        for (name, _, pins), res in zip(jobs, results):
            assert res.returncode != 0 and " failed" in res.stdout, \
                "mutant %r survives pin %s:\n%s" % (name, pins[0], res.stdout[-1500:])
