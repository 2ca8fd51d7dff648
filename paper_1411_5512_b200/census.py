"""Instruction census of the sweep kernels: the numerator of bench.py's alu-pipe roofline.

The persistent sweep kernel is bound by the alu pipe (LOP3 / ISETP / IADD3: the "boolean logic at the bit level" of
PAPER.md:92), so its roofline fraction is

    alu-pipe issue slots used per half-sweep / half-sweep time / measured LOP3 issue rate,

where the slots are the alu-pipe warp instructions PLUS the IMAD.WIDE of Philox and of the address arithmetic: measured
on B200 (ea_selftest_pipes), LOP3 and IMAD.WIDE do not overlap -- any mix of the two issues 0.498 warp instructions per
clock per sub-partition in total, the LOP3 rate alone -- whereas plain 32-bit IMAD does overlap with LOP3.

The instruction count is a property of the BUILT kernel (it includes the data-dependent rare branch, so it is
counted by ncu, `sm__inst_executed_pipe_alu.sum`, not read off the SASS).  It is stored in `alu_census.json` next
to this file together with a SHA-256 of the machine code (SASS) of the sweep kernels in libea_b200.so and of their
source files; `lookup()` refuses a census that matches neither, so a changed kernel can never be credited with an
old count (a comment-only edit changes the source hash but not the SASS).

Refresh after changing a sweep kernel (on a B200, then here):

    gpurun -- 'python bench.py --steps 1 --warmup 3 --sweeps-per-step 200 --no-cpu-baseline --no-next-rows \
               > gpurun_out/plain.log 2>&1 &&
               ncu --clock-control none -k regex:k_sweep_resident -s 3 -c 1 --metrics <METRICS> --csv \
                   --log-file gpurun_out/census.csv python bench.py --steps 1 --warmup 3 --sweeps-per-step 200 \
                   --no-cpu-baseline --no-next-rows'
    python -m paper_1411_5512_b200.census gpurun_out/census.csv 400 profiles/<summary>.md

(400 = half-sweeps of the captured launch.)  This module holds no arithmetic of the method.
"""
import csv
import hashlib
import json
import os
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
CENSUS_PATH = os.path.join(HERE, "alu_census.json")
# every file whose text ends up in the sweep kernels
KERNEL_SOURCES = ["csrc/ea_sweep_resident.cu", "csrc/ea_sweep.cu", "csrc/ea_sweep_common.cuh", "csrc/ea_device.cuh"]
METRICS = ("sm__inst_executed_pipe_alu.sum,sm__inst_executed_pipe_fma.sum,sm__inst_executed_pipe_lsu.sum,"
           "smsp__inst_executed.sum,dram__bytes_read.sum,dram__bytes_write.sum,gpu__time_duration.sum,"
           "sm__pipe_alu_cycles_active.avg.pct_of_peak_sustained_active,"
           "smsp__issue_active.avg.pct_of_peak_sustained_active,launch__registers_per_thread,launch__grid_size,"
           "sm__pipe_fmaheavy_cycles_active.sum,sm__pipe_fmaheavy_cycles_active.avg.pct_of_peak_sustained_elapsed,"
           "sm__cycles_elapsed.sum,smsp__cycles_elapsed.sum,sm__pipe_alu_cycles_active.sum")


def source_hash():
    h = hashlib.sha256()
    for rel in KERNEL_SOURCES:
        with open(os.path.join(HERE, rel), "rb") as f:
            h.update(rel.encode() + b"\0" + f.read() + b"\0")
    return h.hexdigest()


def sass_hash(lib_path=None, pattern="k_sweep_resident"):
    """SHA-256 of the SASS of every function of the built library whose name contains `pattern` (None if cuobjdump is
    not available).  Instruction text only: addresses and encodings included, headers not."""
    import re
    import subprocess
    lib_path = lib_path or os.path.join(HERE, "libea_b200.so")
    try:
        out = subprocess.run(["cuobjdump", "-sass", lib_path], capture_output=True, text=True, timeout=300).stdout
    except (OSError, subprocess.SubprocessError):
        return None
    h, keep, n = hashlib.sha256(), False, 0
    for line in out.splitlines():
        m = re.match(r"\s*Function : (\S+)", line)
        if m:
            keep = pattern in m.group(1)
            if keep:
                h.update(m.group(1).encode() + b"\n")
                n += 1
            continue
        if keep and "/*" in line:
            h.update(line.strip().encode() + b"\n")
    return h.hexdigest() if n else None


def lookup(kernel_key):
    """The census entry of `kernel_key` ("resident_u32_rare", ...) or (None, reason) if absent or stale."""
    try:
        with open(CENSUS_PATH) as f:
            data = json.load(f)
    except (OSError, ValueError):
        return None, "no alu_census.json"
    entry = data.get("kernels", {}).get(kernel_key)
    if entry is None:
        return None, "no census for kernel %r" % kernel_key
    if entry.get("source_sha256") == source_hash():
        return entry, "ok (source hash)"
    sh = sass_hash()
    if sh is not None and entry.get("sass_sha256") == sh:
        return entry, "ok (SASS hash)"
    return None, "census of %r is stale: the kernel changed since it was taken (re-run ncu, see census.py)" % kernel_key


def _num(x):
    return float(str(x).replace(",", ""))


def parse_ncu_csv(path):
    """{metric: value} of the first captured launch in an `ncu --csv` log (long format: one row per metric)."""
    rows = []
    with open(path, newline="") as f:
        lines = [ln for ln in f if not ln.startswith("==")]
    for row in csv.DictReader(lines):
        rows.append(row)
    out, first_id = {}, None
    for row in rows:
        if first_id is None:
            first_id = row.get("ID")
        if row.get("ID") != first_id:
            continue
        name, val, unit = row.get("Metric Name"), row.get("Metric Value"), row.get("Metric Unit", "")
        try:
            v = _num(val)
        except (TypeError, ValueError):
            continue
        scale = {"Kbyte": 1e3, "Mbyte": 1e6, "Gbyte": 1e9, "byte": 1.0, "usecond": 1e-6, "msecond": 1e-3,
                 "nsecond": 1e-9, "ns": 1e-9, "us": 1e-6, "ms": 1e-3, "second": 1.0}.get(unit, 1.0)
        out[name] = v * scale
        out.setdefault("_kernel", row.get("Kernel Name"))
    return out


def kernel_key_of(name):
    """ncu kernel name -> census key, e.g. 'k_sweep_resident<16, unsigned int, 0, 1, 0>(ResidentArgs)' (compute warps, bond
    word, ALWAYS, RARE, HB) -> 'resident_u32_rare'."""
    n = name.replace(" ", "").replace("(bool)", "").replace("(int)", "")
    if "k_sweep_resident" in n:
        inner = n[n.index("<") + 1:n.rindex(">")] if "<" in n else ""
        args = inner.split(",")
        bond = "u32" if "unsignedint" in n else "u64"
        flags = [a in ("1", "true") for a in args[-3:]] if len(args) >= 5 else []
        kind = "heatbath" if len(flags) == 3 and flags[2] else "always" if flags and flags[0] else \
            "rare" if len(flags) >= 2 and flags[1] else "predicated"
        return "resident_%s_%s" % (bond, kind)
    return n.split("<")[0].split("::")[-1]


def main(argv):
    if len(argv) < 3:
        sys.stderr.write(__doc__)
        return 2
    path, half_sweeps = argv[1], float(argv[2])
    profile = argv[3] if len(argv) > 3 else None
    m = parse_ncu_csv(path)
    key = kernel_key_of(m["_kernel"])
    entry = {
        "kernel": m["_kernel"],
        "half_sweeps_in_captured_launch": half_sweeps,
        "alu_warp_inst_per_half_sweep": m["sm__inst_executed_pipe_alu.sum"] / half_sweeps,
        # IMAD.WIDE takes an alu-pipe issue slot as well (ea_selftest_pipes, measured): 4 fmaheavy cycles against 2 of a
        # plain IMAD, so  n_wide = (fmaheavy cycles - 2 x fma-pipe instructions) / 2
        "imad_wide_warp_inst_per_half_sweep": max(0.0, (m.get("sm__pipe_fmaheavy_cycles_active.sum", 0.0)
                                                       - 2.0 * m.get("sm__inst_executed_pipe_fma.sum", 0.0)) / 2.0) / half_sweeps,
        "fma_warp_inst_per_half_sweep": m.get("sm__inst_executed_pipe_fma.sum", 0.0) / half_sweeps,
        "lsu_warp_inst_per_half_sweep": m.get("sm__inst_executed_pipe_lsu.sum", 0.0) / half_sweeps,
        "warp_inst_per_half_sweep": m.get("smsp__inst_executed.sum", 0.0) / half_sweeps,
        "dram_bytes_per_launch": m.get("dram__bytes_read.sum", 0.0) + m.get("dram__bytes_write.sum", 0.0),
        "us_per_half_sweep_under_ncu": 1e6 * m.get("gpu__time_duration.sum", 0.0) / half_sweeps,
        "registers_per_thread": m.get("launch__registers_per_thread"),
        "grid": m.get("launch__grid_size"),
        "source_sha256": source_hash(),
        "sass_sha256": sass_hash(),
        "profile": profile,
        "how": "ncu --metrics (census.METRICS) on one launch of the bench configuration; see census.py",
    }
    entry["alu_slot_warp_inst_per_half_sweep"] = (entry["alu_warp_inst_per_half_sweep"]
                                                  + entry["imad_wide_warp_inst_per_half_sweep"])
    try:
        with open(CENSUS_PATH) as f:
            data = json.load(f)
    except (OSError, ValueError):
        data = {"kernels": {}}
    data["kernels"][key] = entry
    with open(CENSUS_PATH, "w") as f:
        json.dump(data, f, indent=1, sort_keys=True)
        f.write("\n")
    print(key, json.dumps(entry, indent=1))
    return 0


if __name__ == "__main__":
    sys.exit(main(sys.argv))
