"""Turn Nsight Compute CSV exports of `bench.py` runs into the tracked summaries under profiles/.

  python ncu_summary.py step RAW.csv --workload NAME --tag r2b --command "ncu ..."
      RAW.csv = `ncu -i REPORT.ncu-rep --page raw --csv` of an `ncu --set full` capture of one fwd+bwd step.
      Writes profiles/<tag>_step_<workload>.md (one line per launch: time, DRAM bytes, throughputs, tensor-pipe activity)
      and records dram__bytes_read.sum + dram__bytes_write.sum per launch of every GEMM stage in profiles/traffic.json,
      which bench.py reports as roofline.traffic.
  python ncu_summary.py launches LAUNCHES.csv --tag r2b --command "ncu ..."
      LAUNCHES.csv = the `--metrics gpu__time_duration.sum --csv --log-file` launch list.  Writes profiles/<tag>_launches.md.

Reads text files only; runs nothing on a GPU."""
from __future__ import annotations

import argparse
import collections
import csv
import json
import os
import re

ROOT = os.path.dirname(os.path.abspath(__file__))
PROFILES = os.path.join(ROOT, "profiles")
TIME = {"ns": 1e-3, "nsecond": 1e-3, "us": 1.0, "usecond": 1.0, "ms": 1e3, "msecond": 1e3, "s": 1e6, "second": 1e6}
BYTES = {"byte": 1.0, "Kbyte": 1e3, "Mbyte": 1e6, "Gbyte": 1e9, "Tbyte": 1e12}
TC_MODES = {0: "TC_FWD", 1: "TC_FWD_SWIGLU", 2: "TC_DGRAD", 3: "TC_DGRAD_SWIGLU", 4: "TC_WGRAD", 5: "TC_FWD_F32"}
F8_MODES = {0: "F8_FWD", 1: "F8_FWD_SWIGLU", 2: "F8_DGRAD", 3: "F8_DGRAD_SWIGLU"}
# GEMM stage of bench.py's table <- (kernel, mode); the shared expert's single-group launches are told apart by traffic
STAGE_OF = {("tc", 1): "gemm1_swiglu", ("tc", 0): "gemm2", ("tc", 3): "dgrad_down_swiglu", ("tc", 2): "dgrad_gateup",
            ("tc", 4): "wgrad", ("f8", 1): "gemm1_swiglu", ("f8", 0): "gemm2", ("f8", 3): "dgrad_down_swiglu",
            ("f8", 2): "dgrad_gateup"}


def short_name(full):
    n = re.sub(r"\(anonymous namespace\)::|unnamed>::|moe::|^void ", "", full)
    n = re.sub(r"\(.*$", "", n).strip()
    m = re.match(r"(tc|f8)_gemm_kernel<(\d+)(.*)>", n)
    if m:
        kind, mode = m.group(1), int(m.group(2))
        n += " " + (TC_MODES if kind == "tc" else F8_MODES).get(mode, "?")
        return n, (kind, mode)
    return n, None


def read_raw(path):
    rows = list(csv.reader(open(path, newline="")))
    hi = next(i for i, r in enumerate(rows) if r and r[0] == "ID")
    hdr, units = rows[hi], rows[hi + 1]
    return [{h: (v, u) for h, v, u in zip(hdr, r, units)} for r in rows[hi + 2:] if len(r) == len(hdr)]


def val(cell, table=None):
    try:
        v = float(cell[0].replace(",", ""))
    except (ValueError, AttributeError):
        return float("nan")
    return v * table.get(cell[1], 1.0) if table else v


def cmd_step(a):
    rows = read_raw(a.csv)
    out = [f"# {a.tag}: `ncu --set full` capture of one whole fwd+bwd step, {a.workload}", "",
           "Command (on the B200 box, after the same bench command exited 0 without ncu); the CSV was exported on the box with",
           "`ncu -i REPORT.ncu-rep --page raw --csv` and summarised here by `python ncu_summary.py step`:", "",
           "```", a.command, "```", "",
           "| # | kernel | time us | dram read MB | dram write MB | dram thr % | L2 thr % | tensor pipe active % | regs | grid |",
           "|---|---|---|---|---|---|---|---|---|---|"]
    total = 0.0
    per_stage = collections.defaultdict(list)
    for i, r in enumerate(rows):
        name, key = short_name(r["Kernel Name"][0])
        t = val(r["gpu__time_duration.sum"], TIME)
        rd, wr = val(r["dram__bytes_read.sum"], BYTES), val(r["dram__bytes_write.sum"], BYTES)
        total += t
        nan = ("nan", "")
        tp = r.get("sm__pipe_tensor_cycles_active.avg.pct_of_peak_sustained_active") or \
            r.get("sm__inst_executed_pipe_tensor.avg.pct_of_peak_sustained_active") or nan
        out.append(f"| {i} | `{name}` | {t:.1f} | {rd / 1e6:.1f} | {wr / 1e6:.1f} | "
                   f"{val(r.get('gpu__dram_throughput.avg.pct_of_peak_sustained_elapsed', nan)):.1f} | "
                   f"{val(r.get('lts__throughput.avg.pct_of_peak_sustained_elapsed', nan)):.1f} | {val(tp):.1f} | "
                   f"{r['launch__registers_per_thread'][0]} | {r['launch__grid_size'][0]} |")
        if key in STAGE_OF:
            per_stage[STAGE_OF[key]].append(rd + wr)
    out += ["", f"Sum of the {len(rows)} launches: {total:.0f} us (serialised, cold cache, SM clocks not locked: compare SHARES with the",
            "CUDA-event stage table of the bench line, not absolutes)."]
    if a.note:
        out += ["", a.note]
    path = os.path.join(a.out_dir, f"{a.tag}_step_{a.workload}.md")
    open(path, "w").write("\n".join(out) + "\n")
    # traffic per launch of each GEMM stage: the routed experts' launches are the heavy ones (wgrad: three of them)
    stages = {}
    for st, v in per_stage.items():
        v = sorted(v, reverse=True)
        n = 3 if st == "wgrad" else 1
        stages[st] = sum(v[:n]) / len(v[:n])
    tpath = os.path.join(a.out_dir, "traffic.json")
    try:
        rec = json.load(open(tpath))
    except (OSError, ValueError):
        rec = {}
    rec[a.workload] = {"source": f"profiles/{a.tag}_step_{a.workload}.md (ncu --set full, dram__bytes_read.sum + dram__bytes_write.sum per launch)",
                       "stages": stages}
    json.dump(rec, open(tpath, "w"), indent=1, sort_keys=True)
    print(path, tpath)


def cmd_launches(a):
    rows = list(csv.reader(open(a.csv, newline="")))
    hi = next(i for i, r in enumerate(rows) if r and r[0] == "ID")
    hdr = rows[hi]
    ki, mi, ui = hdr.index("Kernel Name"), hdr.index("Metric Value"), hdr.index("Metric Unit")
    agg = collections.OrderedDict()
    for r in rows[hi + 1:]:
        if len(r) <= mi:
            continue
        name, _ = short_name(r[ki])
        agg.setdefault(name, []).append(float(r[mi].replace(",", "")) * TIME.get(r[ui], 1.0))
    n = sum(len(v) for v in agg.values())
    tot = sum(sum(v) for v in agg.values())
    out = [f"# {a.tag}: ncu launch list of one bench run, {a.workload}", "",
           "Command (on the B200 box, after the same command exited 0 without ncu):", "", "```", a.command, "```", "",
           f"{n} launches.  Cold-cache, serialised: compare SHARES.", "", "| kernel | launches | avg us | share of all launches |",
           "|---|---|---|---|"]
    for k, v in agg.items():
        out.append(f"| `{k}` | {len(v)} | {sum(v) / len(v):.1f} | {100 * sum(v) / tot:.1f}% |")
    if a.note:
        out += ["", a.note]
    path = os.path.join(a.out_dir, f"{a.tag}_launches_{a.workload}.md")
    open(path, "w").write("\n".join(out) + "\n")
    print(path)


def main(argv=None):
    ap = argparse.ArgumentParser(description=__doc__, formatter_class=argparse.RawDescriptionHelpFormatter)
    sub = ap.add_subparsers(dest="cmd", required=True)
    for name, fn in (("step", cmd_step), ("launches", cmd_launches)):
        p = sub.add_parser(name)
        p.add_argument("csv")
        p.add_argument("--workload", default="qwen3_30b_a3b_like")
        p.add_argument("--tag", required=True)
        p.add_argument("--command", required=True)
        p.add_argument("--note", default="")
        p.add_argument("--out-dir", default=PROFILES)
        p.set_defaults(fn=fn)
    a = ap.parse_args(argv)
    a.fn(a)


if __name__ == "__main__":
    main()
