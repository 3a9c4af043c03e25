"""Turn an ncu launch list (`ncu --metrics ... --csv --log-file X.csv python bench.py ...`) into the tables kept
under profiles/: one markdown table of the launches grouped by kernel, and profiles/bank_conflicts.json, the
shared-memory bank-conflict counters per kernel that bench.py copies into its JSON line.

    python -m paper_1306_5076_b200.ncu_tables X.csv [Y.csv ...] [--json profiles/bank_conflicts.json] [--source "text"] [--skip N]
                                              [--full profiles/A_full.md ...] [--allow-stale]

--skip N drops the first N launches (the warm-up steps) so that the table describes one timed step.
--full: the committed summaries of `ncu --set full` captures.  A kernel's `excess_per_instruction` in the JSON is the
sum of the "excessive" column of that kernel's per-opcode table there; a kernel without such a capture gets null
(nothing is assumed).  A CSV older than the built libbcf.so is refused (it describes another build) unless
--allow-stale; the JSON records the git commit and the library's build time so that staleness shows.
Reads only the CSV and the .md files; runs nothing on a GPU.
"""
import argparse
import collections
import csv
import json
import os
import re
import subprocess
import sys
import time

CONF_LD = "l1tex__data_bank_conflicts_pipe_lsu_mem_shared_op_ld.sum"
CONF_ST = "l1tex__data_bank_conflicts_pipe_lsu_mem_shared_op_st.sum"
WAVE_LD = "l1tex__data_pipe_lsu_wavefronts_mem_shared_op_ld.sum"
WAVE_ST = "l1tex__data_pipe_lsu_wavefronts_mem_shared_op_st.sum"
TIME = "gpu__time_duration.sum"


def short_name(kernel):
    """`void bcf::pipe::merge_pipe_kernel<bcf::Elem<(int)1, (bool)0>>(...)` -> `merge_pipe_kernel<Elem<1, 0>>`"""
    k = re.sub(r"^void\s+", "", kernel)
    k = re.sub(r">\(.*$", ">", k) if ">(" in k else re.sub(r"\(.*$", "", k)
    k = re.sub(r"\b\w+::", "", k)
    k = re.sub(r"\((int|bool)\)", "", k)
    return k.strip()


def read_launches(path):
    """[(id, kernel, grid, {metric: value})] in launch order."""
    with open(path, newline="") as f:
        lines = [ln for ln in f if ln.startswith('"')]
    launches = collections.OrderedDict()
    for r in csv.DictReader(lines):
        key = int(r["ID"])
        e = launches.setdefault(key, (key, r["Kernel Name"], r["Grid Size"], {}))
        try:
            e[3][r["Metric Name"]] = float(r["Metric Value"].replace(",", ""))
        except ValueError:
            pass
    return list(launches.values())


def group(launches, own_only=True):
    g = collections.OrderedDict()
    for _, kernel, grid, m in launches:
        name = short_name(kernel)
        if own_only and "_kernel" not in name:      # torch's copy / fill kernels between the library's launches
            continue
        e = g.setdefault(name, {"launches": 0, "time_ns": 0.0, "ld": 0.0, "st": 0.0, "wavefronts_ld": 0.0,
                                "wavefronts_st": 0.0, "grid": grid})
        e["launches"] += 1
        e["time_ns"] += m.get(TIME, 0.0)
        e["ld"] += m.get(CONF_LD, 0.0)
        e["st"] += m.get(CONF_ST, 0.0)
        e["wavefronts_ld"] += m.get(WAVE_LD, 0.0)
        e["wavefronts_st"] += m.get(WAVE_ST, 0.0)
    return g


def full_capture_excess(paths):
    """{short kernel name: (sum of excessive shared wavefronts over its LDS / STS instructions, file)} from the
    committed summaries of `ncu --set full` captures (the table under "Per-instruction shared-memory wavefronts")."""
    out = {}
    for path in paths:
        with open(path) as f:
            text = f.read()
        m = re.search(r"^Kernel: `([^`]+)`", text, re.M)
        rows = re.findall(r"^\| ((?:LDS|STS)[\w.]*) \| \d+ \| \d+ \| \d+ \| \d+ \| (\d+) \|$", text, re.M)
        if m and rows:
            out[short_name(m.group(1))] = (sum(int(x) for _, x in rows), os.path.basename(path))
    return out


def build_identity():
    here = os.path.dirname(os.path.abspath(__file__))
    lib = os.path.join(here, "libbcf.so")
    mtime = os.path.getmtime(lib) if os.path.exists(lib) else None
    try:
        head = subprocess.run(["git", "log", "-1", "--format=%h", "--", "paper_1306_5076_b200/csrc", "include"],
                              cwd=os.path.dirname(here), capture_output=True, text=True).stdout.strip()
    except OSError:
        head = ""
    return mtime, {"last_commit_touching_csrc_or_include": head,
                   "libbcf_so_built": time.strftime("%Y-%m-%dT%H:%M:%SZ", time.gmtime(mtime)) if mtime else None}


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("csv", nargs="+")
    ap.add_argument("--json", default=None)
    ap.add_argument("--source", default="")
    ap.add_argument("--skip", type=int, default=0)
    ap.add_argument("--full", nargs="*", default=[])
    ap.add_argument("--allow-stale", action="store_true")
    args = ap.parse_args()
    lib_mtime, identity = build_identity()
    excess = full_capture_excess(args.full)
    out = collections.OrderedDict()
    for path in args.csv:
        if lib_mtime and os.path.getmtime(path) < lib_mtime and not args.allow_stale:
            print("%s is older than libbcf.so: it describes another build (--allow-stale to use it anyway)" % path, file=sys.stderr)
            return 2
        g = group(read_launches(path)[args.skip:])
        total = sum(e["time_ns"] for e in g.values())
        print("\n%s: %d launches of the library's kernels, %.3f ms of kernel time\n"
              % (path, sum(e["launches"] for e in g.values()), total / 1e6))
        print("| kernel | grid | launches | mean time (us) | share of kernel time | ld conflicts | ld wavefronts | st conflicts | st wavefronts |")
        print("|---|---|---|---|---|---|---|---|---|")
        for name, e in g.items():
            k = e["launches"]
            print("| `%s` | %s | %d | %.1f | %.3f | %d (%.1f %%) | %d | %d (%.1f %%) | %d |" % (
                name, e["grid"], k, e["time_ns"] / k / 1e3, e["time_ns"] / total if total else 0.0,
                e["ld"] / k, 100.0 * e["ld"] / max(e["wavefronts_ld"], 1.0), e["wavefronts_ld"] / k,
                e["st"] / k, 100.0 * e["st"] / max(e["wavefronts_st"], 1.0), e["wavefronts_st"] / k))
            out[name] = {"ld": round(e["ld"] / k), "st": round(e["st"] / k), "wavefronts_ld": round(e["wavefronts_ld"] / k),
                         "wavefronts_st": round(e["wavefronts_st"] / k),
                         "excess_per_instruction": excess[name][0] if name in excess else None,
                         "excess_from": excess[name][1] if name in excess else None, "launches_captured": k}
    if args.json:
        doc = {"source": args.source, "build": identity, "per_launch_means": True,
               "note": "ld / st = l1tex__data_bank_conflicts_pipe_lsu_mem_shared_op_{ld,st}.sum per launch; "
                       "excess_per_instruction = sum over the kernel's LDS/STS of (L1 wavefronts shared - ideal) on the source "
                       "page of that kernel's --set full capture (excess_from), null for a kernel with no such capture; "
                       "the kernel-level counters are not per-instruction conflicts but arbitration with the SM's other "
                       "shared-memory and global traffic (profiles/r3_conflict_isolation.md)",
               "kernels": out}
        with open(args.json, "w") as f:
            json.dump(doc, f, indent=1)
            f.write("\n")
    return 0


if __name__ == "__main__":
    sys.exit(main())
