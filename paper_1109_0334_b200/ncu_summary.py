"""Text summaries of an Nsight Compute report of this library's kernels.

    python -m paper_1109_0334_b200.ncu_summary REPORT.ncu-rep --name r2_cfg1_f64 \
        [--out-dir profiles] [--kernel-index 0] [--command "ncu ... python bench.py ..."]

reads the report with `ncu -i REPORT --page raw --csv` and `--page source --csv`
and writes, under --out-dir:

  NAME_ncu.csv       key,value rows: the kernel's name, registers, duration, DRAM
                     bytes, pipe utilisation, cycle counts ... and `source_sha`, the
                     hash of the library source the report belongs to.  bench.py reads
                     this file for roofline.traffic and the ncu pipe figures, and
                     drops them when the hash is not that of the source it runs.
  NAME_ncu.md        the same table for people, the opcode mix, and the command
  NAME_hot_sass.txt  SASS rows of the hot loop with execution counts and stall samples

Nothing here is on the product path: it only reformats a profiler report.
"""
import argparse
import csv
import hashlib
import io
import os
import subprocess
import sys
from collections import defaultdict

HERE = os.path.dirname(os.path.abspath(__file__))
ROOT = os.path.dirname(HERE)

METRICS = [
    "gpu__time_duration.sum", "launch__grid_size", "launch__block_size",
    "launch__registers_per_thread", "launch__occupancy_limit_registers",
    "launch__waves_per_multiprocessor",
    "sm__pipe_fp64_cycles_active.avg.pct_of_peak_sustained_active",
    "sm__pipe_fp64_cycles_active.avg.pct_of_peak_sustained_elapsed",
    "sm__inst_executed_pipe_fp64.avg.pct_of_peak_sustained_active",
    "sm__pipe_fma_cycles_active.avg.pct_of_peak_sustained_active",
    "sm__pipe_fma_cycles_active.avg.pct_of_peak_sustained_elapsed",
    "sm__inst_executed_pipe_fma.avg.pct_of_peak_sustained_active",
    "sm__inst_executed_pipe_alu.avg.pct_of_peak_sustained_active",
    "sm__inst_executed_pipe_xu.avg.pct_of_peak_sustained_active",
    "sm__inst_executed_pipe_lsu.avg.pct_of_peak_sustained_active",
    "smsp__issue_active.avg.pct_of_peak_sustained_active", "smsp__inst_executed.sum",
    "sm__cycles_active.avg", "sm__cycles_elapsed.avg", "sm__cycles_elapsed.avg.per_second",
    "sm__warps_active.avg.per_cycle_active", "smsp__warps_eligible.avg.per_cycle_active",
    "smsp__average_warp_latency_per_inst_issued.ratio",
    "smsp__average_warps_issue_stalled_wait_per_issue_active.ratio",
    "smsp__average_warps_issue_stalled_math_pipe_throttle_per_issue_active.ratio",
    "smsp__average_warps_issue_stalled_not_selected_per_issue_active.ratio",
    "smsp__average_warps_issue_stalled_short_scoreboard_per_issue_active.ratio",
    "smsp__average_warps_issue_stalled_long_scoreboard_per_issue_active.ratio",
    "smsp__average_warps_issue_stalled_dispatch_stall_per_issue_active.ratio",
    "smsp__average_warps_issue_stalled_branch_resolving_per_issue_active.ratio",
    "smsp__average_warps_issue_stalled_barrier_per_issue_active.ratio",
    "smsp__average_warps_issue_stalled_no_instruction_per_issue_active.ratio",
    "dram__bytes_read.sum", "dram__bytes_write.sum",
    "dram__throughput.avg.pct_of_peak_sustained_elapsed",
    "sm__throughput.avg.pct_of_peak_sustained_elapsed",
]

BYTE_UNITS = {"byte": 1.0, "Kbyte": 1e3, "Mbyte": 1e6, "Gbyte": 1e9}
TIME_UNITS = {"ns": 1e-6, "us": 1e-3, "ms": 1.0, "s": 1e3,
              "nsecond": 1e-6, "usecond": 1e-3, "msecond": 1.0, "second": 1e3}


def source_sha():
    """Hash of the library source (csrc/* and include/afm.h), in sorted file order."""
    h = hashlib.sha256()
    files = sorted(os.path.join(HERE, "csrc", f) for f in os.listdir(os.path.join(HERE, "csrc")))
    files.append(os.path.join(ROOT, "include", "afm.h"))
    for f in files:
        h.update(os.path.basename(f).encode())
        h.update(open(f, "rb").read())
    return h.hexdigest()[:16]


def _ncu_csv(rep, page):
    out = subprocess.run(["ncu", "-i", rep, "--page", page, "--csv"], capture_output=True,
                         text=True, check=True).stdout
    return list(csv.reader(io.StringIO(out)))


def read_raw(rep, index=0):
    """(kernel name, {metric: (unit, value string)}) of launch `index` of the report."""
    rows = _ncu_csv(rep, "raw")
    hdr, units, data = rows[0], rows[1], rows[2:]
    col = {k: i for i, k in enumerate(hdr)}
    r = data[index]
    vals = {m: (units[col[m]], r[col[m]]) for m in METRICS if m in col and r[col[m]] != ""}
    return r[col["Kernel Name"]], vals


def _num(s):
    return float(s.replace(",", ""))


def to_ms(unit, value):
    return _num(value) * TIME_UNITS[unit]


def to_bytes(unit, value):
    return _num(value) * BYTE_UNITS[unit]


def hot_sass(rep, thr=0.05):
    """(total warp-instructions, [(opcode, count)], [(row, executions, samples, sass)])."""
    rows = _ncu_csv(rep, "source")
    hdr, data = rows[1], rows[2:]
    col = {k: i for i, k in enumerate(hdr)}
    S, EX, SMP = col["Source"], col["Instructions Executed"], col["# Samples"]
    mx = max(int(r[EX] or 0) for r in data)
    ops = defaultdict(int)
    hot = []
    for k, r in enumerate(data):
        ex = int(r[EX] or 0)
        t = r[S].split()
        ops[t[1] if t[0].startswith("@") else t[0]] += ex
        if ex >= thr * mx:
            hot.append((k, ex, r[SMP], r[S].strip()))
    return sum(ops.values()), sorted(ops.items(), key=lambda kv: -kv[1]), hot


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("report")
    ap.add_argument("--name", required=True)
    ap.add_argument("--out-dir", default=os.path.join(ROOT, "profiles"))
    ap.add_argument("--kernel-index", type=int, default=0)
    ap.add_argument("--command", default="")
    ap.add_argument("--title", default="")
    ap.add_argument("--no-sass", action="store_true", help="skip NAME_hot_sass.txt")
    a = ap.parse_args()
    kname, vals = read_raw(a.report, a.kernel_index)
    total, ops, hot = hot_sass(a.report)
    sha = source_sha()
    base = os.path.join(a.out_dir, a.name)
    rows = [("kernel", kname), ("source_sha", sha), ("command", a.command),
            ("duration_ms", "%.6f" % to_ms(*vals["gpu__time_duration.sum"])),
            ("dram_bytes_read", "%d" % to_bytes(*vals["dram__bytes_read.sum"])),
            ("dram_bytes_write", "%d" % to_bytes(*vals["dram__bytes_write.sum"]))]
    rows += [(m, _num(v[1])) for m, v in vals.items()]
    # executed floating-point warp-instructions of the launch (source page): what
    # bench.py turns into executed FLOP/s, SURVEY.md 8(d) definition (2)
    opd = dict(ops)
    for prefix, key in (("D", "fp64"), ("F", "fp32")):
        fma = sum(v for k, v in opd.items() if k.split(".")[0] == prefix + "FMA")
        add = sum(v for k, v in opd.items() if k.split(".")[0] == prefix + "ADD")
        mul = sum(v for k, v in opd.items() if k.split(".")[0] == prefix + "MUL")
        rows += [("executed_%s_fma" % key, fma), ("executed_%s_add" % key, add),
                 ("executed_%s_mul" % key, mul)]
    with open(base + "_ncu.csv", "w", newline="") as f:
        w = csv.writer(f)
        w.writerow(("key", "value"))
        w.writerows(rows)
    md = ["# %s" % (a.title or a.name), "",
          "Command (one B200 under gpurun, repository root; a number printed by a run "
          "under ncu is never a bench value):", "", "```", a.command, "```", "",
          "Summarised with `python -m paper_1109_0334_b200.ncu_summary` "
          "(library source hash `%s`; machine-readable copy: `%s_ncu.csv`)." % (sha, a.name),
          "", "Kernel: `%s`" % kname, "", "| metric | unit | value |", "|---|---|---|"]
    md += ["| %s | %s | %s |" % (m, v[0], v[1]) for m, v in vals.items()]
    md += ["", "Executed warp-instructions by opcode (%d in total):" % total, "",
           "| opcode | warp-instructions | share |", "|---|---|---|"]
    md += ["| %s | %d | %.3f |" % (k, v, v / total) for k, v in ops[:16]]
    if "_q<" in kname:
        md += ["", "(The opcode counts come from ncu's instrumented pass.  A queue worker that "
               "waits sleeps for a time in nanoseconds between two polls, and that pass runs "
               "many times slower than a timed launch: its polling instructions -- "
               "LDG.E.STRONG.GPU, NANOSLEEP, YIELD, CS2R and the BRA / ISETP around them -- "
               "are over-counted here by that factor.  `smsp__inst_executed.sum` above is "
               "from a hardware-counter pass.)"]
    md += ["", "Hot-loop SASS: `%s_hot_sass.txt`." % a.name, ""] if not a.no_sass else [""]
    open(base + "_ncu.md", "w").write("\n".join(md))
    if a.no_sass:
        print("wrote %s_ncu.csv, _ncu.md (kernel %s, %.3f ms)"
              % (base, kname.split("(")[0], to_ms(*vals["gpu__time_duration.sum"])))
        return 0
    with open(base + "_hot_sass.txt", "w") as f:
        f.write("# %s: SASS rows with >= 5%% of the maximum execution count "
                "(ncu --page source)\n# columns: row, warp-level executions, stall samples, "
                "SASS\n" % kname)
        for k, ex, smp, sass in hot:
            f.write("%5d %12d %7s  %s\n" % (k, ex, smp, sass))
    print("wrote %s_ncu.csv, _ncu.md, _hot_sass.txt (kernel %s, %.3f ms)"
          % (base, kname.split("(")[0], to_ms(*vals["gpu__time_duration.sum"])))
    return 0


if __name__ == "__main__":
    sys.exit(main())
