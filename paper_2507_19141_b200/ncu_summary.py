"""Turn an ncu CSV into the per-launch table and the traffic summary that `profiles/` holds and `bench.py` reads.

    ncu -i gpurun_out/prof.ncu-rep --page raw --csv > gpurun_out/prof_raw.csv      # wide: one row per launch
    python -m paper_2507_19141_b200.ncu_summary gpurun_out/prof_raw.csv --config C4 \\
        --command "<the ncu command that made the capture>" --md profiles/ncu_step_r02.md \\
        --traffic profiles/traffic.json

Accepts both CSV shapes ncu writes: the wide `--page raw --csv` export (header row, units row, one row per launch)
and the long `--csv --log-file` list of a `--metrics` run (one row per launch and metric).  Units are normalised
(bytes, microseconds).  The traffic file gets, per config: DRAM bytes (read + write) of every launch class and of
the C-ABI calls of ONE step — "fwd_call" (hash4d_fwd_kernel launches and, under SORT_COARSE, the sort before them),
"bwd_call" (zero_kernel + hash4d_bwd_kernel + hash4d_bwd_runs_kernel launches), "step" (both) — taken from the LAST
complete step in the capture.  No number is typed by hand.
"""
from __future__ import annotations

import argparse
import csv
import json
import os
import re
import sys

WANT = [
    ("gpu__time_duration.sum", "us"),
    ("dram__bytes_read.sum", "MB"),
    ("dram__bytes_write.sum", "MB"),
    ("lts__t_sector_hit_rate.pct", "%"),
    ("lts__throughput.avg.pct_of_peak_sustained_elapsed", "%"),
    ("l1tex__throughput.avg.pct_of_peak_sustained_elapsed", "%"),
    ("l1tex__t_sectors_pipe_lsu_mem_global_op_ld.sum", "sectors"),
    ("l1tex__t_requests_pipe_lsu_mem_global_op_ld.sum", "requests"),
    ("l1tex__t_sectors_pipe_lsu_mem_global_op_red.sum", "sectors"),
    ("l1tex__t_requests_pipe_lsu_mem_global_op_red.sum", "requests"),
    ("sm__warps_active.avg.pct_of_peak_sustained_active", "%"),
    ("launch__registers_per_thread", "regs"),
]

_SCALE = {"byte": 1.0, "Kbyte": 1e3, "Mbyte": 1e6, "Gbyte": 1e9, "Tbyte": 1e12,
          "ns": 1e-3, "us": 1.0, "usecond": 1.0, "ms": 1e3, "msecond": 1e3, "s": 1e6, "second": 1e6, "nsecond": 1e-3}


def _num(text: str):
    try:
        return float(text.replace(",", ""))
    except ValueError:
        return None


def _normalise(name: str, unit: str, value):
    """bytes for byte metrics, microseconds for durations, unchanged otherwise."""
    if value is None:
        return None
    if unit in _SCALE and ("bytes" in name or "duration" in name):
        return value * _SCALE[unit]
    return value


def _short(kernel: str) -> str:
    m = re.search(r"(\w+)\s*(<[^(]*>)?\s*\(", kernel)
    name = m.group(1) if m else kernel
    tmpl = re.search(rf"{name}\s*<([^(]*)>\s*\(", kernel)
    return f"{name}<{tmpl.group(1)}>" if tmpl else name


def read_launches(path: str):
    """-> list of {"id", "kernel", "grid", "block", metric: value...} in launch order."""
    rows = [r for r in csv.reader(l for l in open(path, newline="") if l.startswith('"'))]
    if not rows:
        raise SystemExit(f"{path}: no CSV rows")
    head = rows[0]
    col = {n: i for i, n in enumerate(head)}
    launches = {}
    if "Metric Name" in col:                                           # long format
        for r in rows[1:]:
            lid = int(r[col["ID"]])
            d = launches.setdefault(lid, {"id": lid, "kernel": r[col["Kernel Name"]], "grid": r[col["Grid Size"]],
                                          "block": r[col["Block Size"]]})
            name = r[col["Metric Name"]]
            d[name] = _normalise(name, r[col["Metric Unit"]], _num(r[col["Metric Value"]]))
    else:                                                              # wide format: row 1 = units
        units = rows[1]
        # section prefixes ("SM_A.TriageCompute.") are stripped; the first occurrence of a metric wins
        names = [h.split(".", 2)[2] if h.count(".") >= 3 and h.split(".")[1] == "TriageCompute" else h for h in head]
        for r in rows[2:]:
            if not r[col["ID"]].strip():
                continue
            lid = int(r[col["ID"]])
            d = {"id": lid, "kernel": r[col["Kernel Name"]], "grid": r[col["Grid Size"]], "block": r[col["Block Size"]]}
            for i, n in enumerate(names):
                if i < len(r) and d.get(n) is None:                    # first column that holds a value wins
                    d[n] = _normalise(n, units[i] if i < len(units) else "", _num(r[i]))
            launches[lid] = d
    return [launches[k] for k in sorted(launches)]


_BWD_CALL = ("hash4d_bwd_kernel", "hash4d_bwd_runs_kernel", "zero_kernel")   # launches of one dash_hash4d_bwd call
_SORT = ("sort4d_", "sort_scan_")   # the coarse sort: in the forward call under SORT_COARSE (bench.py), else in bwd


def _is(kernel: str, names) -> bool:
    return any(n in kernel for n in names)


def last_step(launches):
    """The launches of the last complete step.  A step is one forward call — the hash4d_fwd_kernel launch(es), preceded
    under SORT_COARSE by the coarse sort (zero_kernel of its histogram + sort launches) — followed by the launches of
    one backward call (zero / bwd / bwd_runs, and the sort when the backward does its own); it ends where the next
    forward call starts or at anything else.  The last step that holds at least one hash4d_bwd_kernel wins."""
    n = len(launches)
    k = [l["kernel"] for l in launches]
    starts = []                                        # (first launch of the forward call, its first fwd launch)
    for f in range(n):
        if "hash4d_fwd_kernel" in k[f] and (f == 0 or "hash4d_fwd_kernel" not in k[f - 1]):
            s = f
            while s > 0 and _is(k[s - 1], _SORT):
                s -= 1
            if s < f and s > 0 and "zero_kernel" in k[s - 1]:
                s -= 1
            starts.append((s, f))
    for j in range(len(starts) - 1, -1, -1):
        s, f = starts[j]
        limit = starts[j + 1][0] if j + 1 < len(starts) else n
        e = f
        while e < limit and "hash4d_fwd_kernel" in k[e]:
            e += 1
        b = e
        while e < limit and _is(k[e], _BWD_CALL + _SORT):
            e += 1
        if any("hash4d_bwd_kernel" in x for x in k[b:e]):
            return launches[s:e]
    return []


def is_fwd_call(step, i) -> bool:
    """Launch i of `step` belongs to the forward call: the hash4d_fwd_kernel launches and the sort before them."""
    first_bwd = next((j for j, l in enumerate(step) if _is(l["kernel"], ("hash4d_bwd_kernel", "hash4d_bwd_runs_kernel"))),
                     len(step))
    last_fwd = max((j for j, l in enumerate(step) if "hash4d_fwd_kernel" in l["kernel"]), default=-1)
    return i <= last_fwd and i < first_bwd


def dram(l):
    return (l.get("dram__bytes_read.sum") or 0.0) + (l.get("dram__bytes_write.sum") or 0.0)


def markdown(launches, step, title, command):
    out = [f"# {title}", "", "Command:", "", "```", command, "```", "",
           f"{len(launches)} launches captured; the last complete step is launches "
           f"{step[0]['id']}..{step[-1]['id']} ({len(step)} launches).  Written by "
           "`python -m paper_2507_19141_b200.ncu_summary`; nothing below is typed by hand.", "",
           "| # | kernel | grid | " + " | ".join(f"{n.split('.')[0].replace('__', ' ')} [{u}]" for n, u in WANT) + " |",
           "|---|---|---|" + "---|" * len(WANT)]
    for l in step:
        cells = []
        for n, u in WANT:
            v = l.get(n)
            if v is None:
                cells.append("")
            elif u == "MB":
                cells.append(f"{v / 1e6:.1f}")
            elif u in ("us", "%"):
                cells.append(f"{v:.1f}")
            else:
                cells.append(f"{v:.0f}")
        out.append(f"| {l['id']} | `{_short(l['kernel'])}` | {l['grid']} | " + " | ".join(cells) + " |")
    tot_t = sum(l.get("gpu__time_duration.sum") or 0 for l in step)
    fwd = [l for i, l in enumerate(step) if is_fwd_call(step, i)]
    bwd = [l for i, l in enumerate(step) if not is_fwd_call(step, i)]
    out += ["", f"Step totals: {tot_t:.1f} us under ncu (serialised, cold cache — shares, not absolutes); DRAM read+write "
                f"fwd call {sum(map(dram, fwd)) / 1e9:.3f} GB, bwd call {sum(map(dram, bwd)) / 1e9:.3f} GB, step "
                f"{sum(map(dram, step)) / 1e9:.3f} GB.",
            f"Share of the step's time: fwd {sum(l.get('gpu__time_duration.sum') or 0 for l in fwd) / max(tot_t, 1e-9):.3f}, "
            f"bwd + zero {sum(l.get('gpu__time_duration.sum') or 0 for l in bwd) / max(tot_t, 1e-9):.3f}."]
    return "\n".join(out) + "\n"


def main(argv=None):
    ap = argparse.ArgumentParser(description=__doc__, formatter_class=argparse.RawDescriptionHelpFormatter)
    ap.add_argument("csv")
    ap.add_argument("--config", default="C4")
    ap.add_argument("--command", default="(not recorded)")
    ap.add_argument("--title", default=None)
    ap.add_argument("--md", default=None, help="write the per-launch table here")
    ap.add_argument("--traffic", default=None, help="merge the DRAM totals into this JSON file")
    args = ap.parse_args(argv)
    launches = read_launches(args.csv)
    step = last_step(launches)
    if not step:
        raise SystemExit("no complete fwd + bwd step in the capture")
    if args.md:
        with open(args.md, "w") as fh:
            fh.write(markdown(launches, step, args.title or f"ncu per-launch table, one step of {args.config}",
                              args.command))
    fwd = [l for i, l in enumerate(step) if is_fwd_call(step, i)]
    bwd = [l for i, l in enumerate(step) if not is_fwd_call(step, i)]
    summary = {"fwd_call": sum(map(dram, fwd)), "bwd_call": sum(map(dram, bwd)), "step": sum(map(dram, step)),
               "launches_in_step": len(step), "source_csv": os.path.basename(args.csv), "command": args.command}
    if args.traffic:
        data = {}
        if os.path.exists(args.traffic):
            with open(args.traffic) as fh:
                data = json.load(fh)
        data.pop("_source", None)
        data[args.config] = summary
        with open(args.traffic, "w") as fh:
            json.dump(data, fh, indent=1)
            fh.write("\n")
    print(json.dumps(summary))
    return 0


if __name__ == "__main__":
    sys.exit(main())
