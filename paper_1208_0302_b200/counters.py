"""Counted work of a kernel from an ncu report -> an entry of profiles/<round>_counters.json, which bench.py reads.

bench.py's `roofline` needs the EXECUTED FP32 work per wavelength point of the kernel it times.
That number belongs to one build of csrc/ and one workload shape; typed into bench.py it goes stale silently.  This module
writes it from a capture, together with a hash of the sources the captured library was built from, and bench.py refuses
to turn a count into a fraction of peak when that hash is not the hash of the sources it is running.

    ncu --set full --clock-control none --import-source on -k regex:ga_invert -c 1 -o gpurun_out/<name> -f python bench.py ...
    python -m paper_1208_0302_b200.counters --rep gpurun_out/<name>.ncu-rep --key config3_fulldisc/triplets \
        --points <wavelength points of the captured launch> --pixels <pixels of it> --command "<the ncu command>" \
        --out profiles/r2_counters.json

Counting rule (as in profiles/r1i_ga_invert_ncu.md): predicated-on thread instructions per SASS opcode from the source page;
FFMA2 = 4 flop, FMUL2 / FADD2 / FFMA = 2, FMUL / FADD = 1; an FMA-pipe lane-slot = one lane of a packed or scalar FP32
instruction (packed = 2 slots).  No method arithmetic lives here.
"""
import argparse
import csv
import hashlib
import io
import json
import os
import re
import subprocess

HERE = os.path.dirname(os.path.abspath(__file__))
ROOT = os.path.dirname(HERE)
FLOP = {"FFMA2": 4, "FMUL2": 2, "FADD2": 2, "FFMA": 2, "FMUL": 1, "FADD": 1}
SLOTS = {"FFMA2": 2, "FMUL2": 2, "FADD2": 2, "FFMA": 1, "FMUL": 1, "FADD": 1}


# The files the counted kernels (ga_invert_kernel, me_synth_kernel) are compiled from.  Host-side code (me_api.cu: validation and
# descriptors; me_kernels.cu: launch glue and the small hook kernels; me_probe.cu) is deliberately NOT in the hash: an edit
# there cannot change the instruction mix of the counted kernels, and hashing it would mark good counts stale.
KERNEL_SOURCES = ["me_device.cuh", "me_inst.cuh", "faddeeva_table.h", "me_launch.h"]


def csrc_sha():
    """sha256 over KERNEL_SOURCES, the csrc/me_inst_*.cu instantiation units and include/me.h (ME_MAX_* fix the descriptor
    layout), in that order."""
    h = hashlib.sha256()
    d = os.path.join(HERE, "csrc")
    inst = sorted(f for f in os.listdir(d) if f.startswith("me_inst_") and f.endswith(".cu"))
    for f in [os.path.join(d, f) for f in KERNEL_SOURCES + inst] + [os.path.join(ROOT, "include", "me.h")]:
        h.update(os.path.basename(f).encode())
        h.update(open(f, "rb").read())
    return h.hexdigest()[:16]


def _ncu_csv(rep, page):
    out = subprocess.run(["ncu", "-i", rep, "--page", page, "--csv"], capture_output=True, text=True, check=True).stdout
    return list(csv.reader(io.StringIO(out)))


def opcode_counts(rep):
    """{opcode: predicated-on thread instructions} of the (single) kernel in the report's source page."""
    rows = _ncu_csv(rep, "source")
    hdr_i = next(i for i, r in enumerate(rows) if r and r[0] == "Address")
    hdr = rows[hdr_i]
    c_src, c_thr = hdr.index("Source"), hdr.index("Predicated-On Thread Instructions Executed")
    kernel = rows[0][1] if rows and rows[0] and rows[0][0] == "Kernel Name" else ""
    counts = {}
    for r in rows[hdr_i + 1:]:
        if len(r) <= c_thr:
            continue
        m = re.match(r"\s*(?:@!?U?P\d+\s+)?([A-Z][A-Z0-9_]*)", r[c_src])       # strip the predicate, keep the base opcode
        if not m:
            continue
        try:
            n = int(float(r[c_thr].replace(",", "")))
        except ValueError:
            continue
        counts[m.group(1)] = counts.get(m.group(1), 0) + n
    return kernel, counts


def raw_metrics(rep, names):
    rows = _ncu_csv(rep, "raw")
    hdr, vals = rows[0], rows[2]
    out = {}
    for n in names:
        if n in hdr:
            try:
                out[n] = float(vals[hdr.index(n)].replace(",", ""))
            except ValueError:
                out[n] = None
    units = {n: rows[1][hdr.index(n)] for n in names if n in hdr}
    return out, units


def _bytes(v, unit):
    scale = {"byte": 1.0, "Kbyte": 1e3, "Mbyte": 1e6, "Gbyte": 1e9, "Tbyte": 1e12}
    return None if v is None else v * scale.get(unit, 1.0)


def entry_from_report(rep, points, pixels, command, sha=None):
    """sha: the csrc_sha the CAPTURED process printed (bench.py's JSON line carries it); default = the tree as it stands."""
    kernel, counts = opcode_counts(rep)
    total = sum(counts.values())
    flop = sum(FLOP[k] * counts.get(k, 0) for k in FLOP)
    slots = sum(SLOTS[k] * counts.get(k, 0) for k in SLOTS)
    names = ["gpu__time_duration.sum", "launch__registers_per_thread", "dram__bytes_read.sum", "dram__bytes_write.sum",
             "sm__pipe_fma_cycles_active.avg.pct_of_peak_sustained_elapsed", "sm__pipe_fma_cycles_active.avg.pct_of_peak_sustained_active",
             "smsp__issue_active.avg.pct_of_peak_sustained_active", "smsp__thread_inst_executed_per_inst_executed.ratio"]
    m, u = raw_metrics(rep, names)
    dram = (_bytes(m.get("dram__bytes_read.sum"), u.get("dram__bytes_read.sum")) or 0.0) + \
           (_bytes(m.get("dram__bytes_write.sum"), u.get("dram__bytes_write.sum")) or 0.0)
    return {"kernel": kernel, "csrc_sha": sha or csrc_sha(), "report": os.path.basename(rep), "command": command,
            "captured_points": int(points), "captured_pixels": int(pixels),
            "flop_per_lambda_point": flop / points, "fma_lane_slots_per_lambda_point": slots / points,
            "mufu_per_lambda_point": counts.get("MUFU", 0) / points, "thread_inst_per_lambda_point": total / points,
            "per_point": {k: counts.get(k, 0) / points for k in list(FLOP) + ["MUFU"]},
            "fma_pipe_busy_elapsed": (m.get("sm__pipe_fma_cycles_active.avg.pct_of_peak_sustained_elapsed") or 0.0) / 100.0,
            "issue_active": (m.get("smsp__issue_active.avg.pct_of_peak_sustained_active") or 0.0) / 100.0,
            "threads_per_warp_inst": m.get("smsp__thread_inst_executed_per_inst_executed.ratio"),
            "registers_per_thread": m.get("launch__registers_per_thread"),
            "duration_ncu": m.get("gpu__time_duration.sum"), "duration_unit": u.get("gpu__time_duration.sum"),
            "dram_bytes_per_pixel": dram / pixels if pixels else None}


def load(path=None):
    """The newest profiles/r*_counters.json (or `path`): ({key: entry}, path relative to the repo).  ({}, None) if none."""
    if path is None:
        d = os.path.join(ROOT, "profiles")
        c = sorted(f for f in os.listdir(d) if re.match(r"r\d+\w*_counters\.json$", f)) if os.path.isdir(d) else []
        if not c:
            return {}, None
        path = os.path.join(d, c[-1])
    return json.load(open(path)), os.path.relpath(path, ROOT)


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--rep", required=True)
    ap.add_argument("--key", required=True, help="<workload name>/<triplets|full>, e.g. config3_fulldisc/triplets")
    ap.add_argument("--points", type=float, required=True, help="wavelength points of the captured launch")
    ap.add_argument("--pixels", type=float, required=True, help="pixels (or vectors) of the captured launch")
    ap.add_argument("--command", default="")
    ap.add_argument("--csrc-sha", default=None, help="csrc_sha printed by the captured bench.py run (default: the tree as it stands)")
    ap.add_argument("--out", required=True)
    a = ap.parse_args()
    data = json.load(open(a.out)) if os.path.exists(a.out) else {}
    data[a.key] = entry_from_report(a.rep, a.points, a.pixels, a.command, a.csrc_sha)
    with open(a.out, "w") as fh:
        json.dump(data, fh, indent=1, sort_keys=True)
        fh.write("\n")
    print(json.dumps(data[a.key], indent=1))


if __name__ == "__main__":
    main()
