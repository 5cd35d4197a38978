"""Turn Nsight Compute CSV output into the text summaries under profiles/ (no GPU needed).

    # launch list (ncu --metrics gpu__time_duration.sum --csv --log-file launches.csv <cmd>)
    python -m paper_2602_17938_b200.ncu_summary launches gpurun_out/r03_launches.csv --out profiles/r03_launches.md \
        --command "<the ncu command>"

    # full capture (ncu --set full -o full <cmd>;  ncu -i full.ncu-rep --page raw --csv > full_raw.csv)
    python -m paper_2602_17938_b200.ncu_summary full gpurun_out/r03_full_raw.csv --out profiles/r03_ncu_full.md \
        --command "<the ncu command>" --traffic profiles/ncu_traffic.json --traffic-key noise_S --traffic-kernel k_noise_S_tma

The full summary carries, per launch, the achieved DRAM rate in GB/s (dram__bytes_read.sum + dram__bytes_write.sum over
gpu__time_duration.sum) against both the measured copy bandwidth of this pool's B200s (MEASURED_PEAKS.json, else the
fallback of B200_PROFILING.md) and the ~8 TB/s nominal figure BASELINE.json's north_star quotes.  --traffic writes the
dram bytes of the first launch whose name contains --traffic-kernel into a small JSON file that bench.py reads for the
`roofline.traffic` field (so that figure is a captured number, not a typed-in constant).

Only csv / json / re from the standard library; nothing here is on the product path.
"""
from __future__ import annotations

import argparse
import csv
import io
import json
import os
import re
import sys

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
NOMINAL_HBM_GBS = 8000.0          # BASELINE.json north_star: "against B200's ~8 TB/s"
FALLBACK_HBM_GBS = 6650.0         # B200_PROFILING.md fallback when MEASURED_PEAKS.json is absent

UNIT_BYTES = {"byte": 1.0, "Kbyte": 1e3, "Mbyte": 1e6, "Gbyte": 1e9, "Tbyte": 1e12}
UNIT_SECONDS = {"ns": 1e-9, "nsecond": 1e-9, "us": 1e-6, "usecond": 1e-6, "ms": 1e-3, "msecond": 1e-3, "s": 1.0,
                "second": 1.0}


def measured_hbm_gbs():
    path = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(path):
        return float(json.load(open(path))["hbm_gbs"]), "MEASURED_PEAKS.json"
    return FALLBACK_HBM_GBS, "fallback of B200_PROFILING.md"


def _rows(path):
    """CSV rows of an ncu log: everything from the header line (the one that starts with "ID") on."""
    text = open(path, newline="").read()
    start = text.find('"ID"')
    if start < 0:
        raise SystemExit("%s: no ncu CSV header found" % path)
    return list(csv.reader(io.StringIO(text[start:])))


def _num(s):
    s = s.replace(",", "").strip()
    try:
        return float(s)
    except ValueError:
        return None


def short_name(k):
    """lac::k_noise_S_tma<7>(CUtensorMap, ...) -> k_noise_S_tma<7>"""
    k = re.sub(r"^(void\s+)?", "", k.strip())
    k = k.split("(")[0]
    return re.sub(r"^(lac::|\(anonymous namespace\)::)+", "", k)


# ------------------------------------------------------------------------------------------- launch list
def launches(args):
    rows = _rows(args.csv)
    head = rows[0]
    col = {n: i for i, n in enumerate(head)}
    out = []          # (kernel, grid, block, us)
    if "Metric Name" in col:                     # long format: one row per (launch, metric)
        for r in rows[1:]:
            if len(r) <= col["Metric Value"] or r[col["Metric Name"]] != "gpu__time_duration.sum":
                continue
            v = _num(r[col["Metric Value"]])
            unit = r[col["Metric Unit"]] if "Metric Unit" in col else "ns"
            out.append((short_name(r[col["Kernel Name"]]), r[col["Grid Size"]], r[col["Block Size"]],
                        v * UNIT_SECONDS.get(unit, 1e-9) * 1e6))
    else:                                        # raw format: one row per launch, units in the second row
        units = rows[1]
        i = col["gpu__time_duration.sum"]
        for r in rows[2:]:
            if len(r) > i and _num(r[i]) is not None:
                out.append((short_name(r[col["Kernel Name"]]), r[col["Grid Size"]], r[col["Block Size"]],
                            _num(r[i]) * UNIT_SECONDS.get(units[i], 1e-9) * 1e6))
    mine = [o for o in out if o[0].startswith("k_")]
    other = [o for o in out if not o[0].startswith("k_")]
    head_n = args.head if args.head > 0 else len(mine)

    def table(part):
        per = {}
        for k, g, b, us in part:
            d = per.setdefault(k, dict(n=0, us=0.0, grids=set()))
            d["n"] += 1
            d["us"] += us
            d["grids"].add("%s x %s" % (g, b))
        total = sum(d["us"] for d in per.values()) or 1.0
        T = ["| kernel | grid x block | launches | avg us | total us | share of the library's kernel time |", "|---|---|---|---|---|---|"]
        for k, d in sorted(per.items(), key=lambda kv: -kv[1]["us"]):
            T.append("| %s | %s | %d | %.1f | %.1f | %.3f |" % (k, "; ".join(sorted(d["grids"])), d["n"], d["us"] / d["n"], d["us"],
                                                               d["us"] / total))
        return T, total

    L = ["# %s -- ncu launch list" % args.label, "", "Command (under gpurun, after the same command exited 0 without ncu):", "",
         "    " + args.command, "",
         "Made from the CSV by `python -m paper_2602_17938_b200.ncu_summary launches`.  Per-launch times under ncu are",
         "cold-cache and serialised: compare SHARES with bench.py's `kernel_share_of_step`, not absolutes.", ""]
    T, total = table(mine[:head_n])
    if args.head > 0:
        L += ["The first %d launches of the library's kernels (%s):" % (head_n, args.head_what), ""]
    L += T
    L += ["", "%d launches, %.1f us in total%s." % (min(head_n, len(mine)), total,
                                                    (" = %.1f us per frame" % (total * args.frame_launches / head_n))
                                                    if args.head > 0 and args.frame_launches > 0 else "")]
    if args.frame_launches > 0 and len(mine) >= args.frame_start + args.frame_launches:
        a = args.frame_start
        L += ["", "One frame, launch by launch (us), launches %d-%d:" % (a, a + args.frame_launches - 1), "", "```"]
        L += ["%-28s %-20s %8.1f" % (k, g, us) for k, g, b, us in mine[a:a + args.frame_launches]]
        L += ["```", "", "Sum: %.1f us." % sum(o[3] for o in mine[a:a + args.frame_launches])]
    if head_n < len(mine):
        T2, total2 = table(mine[head_n:])
        L += ["", "The other %d launches of the library's kernels captured by the same command (%s):" % (len(mine) - head_n, args.rest_what), ""]
        L += T2
    L += ["", "%d launches that are not the library's (%s)." % (len(other), ", ".join(sorted({o[0][:40] for o in other})) or "none")]
    open(args.out, "w").write("\n".join(L) + "\n")
    print("wrote", args.out)


# ------------------------------------------------------------------------------------------- full capture
WANTED = [    # (column title, candidate metric names, format)
    ("regs", ["launch__registers_per_thread"], "%d"),
    ("warps active %", ["sm__warps_active.avg.pct_of_peak_sustained_active"], "%.1f"),
    ("issue active %", ["sm__inst_issued.avg.pct_of_peak_sustained_active", "smsp__issue_active.avg.pct_of_peak_sustained_active",
                        "sm__issue_active.avg.pct_of_peak_sustained_active"], "%.1f"),
    ("alu pipe %", ["sm__inst_executed_pipe_alu.avg.pct_of_peak_sustained_active",
                    "sm__pipe_alu_cycles_active.avg.pct_of_peak_sustained_active"], "%.1f"),
    ("fma pipe %", ["sm__inst_executed_pipe_fma.avg.pct_of_peak_sustained_active",
                    "sm__pipe_fma_cycles_active.avg.pct_of_peak_sustained_active"], "%.1f"),
    ("lsu pipe %", ["sm__inst_executed_pipe_lsu.avg.pct_of_peak_sustained_active"], "%.1f"),
    ("dram % (ncu)", ["gpu__dram_throughput.avg.pct_of_peak_sustained_elapsed"], "%.1f"),
    ("warp inst", ["smsp__inst_executed.sum", "sm__inst_executed.sum"], "%d"),
]


def full(args):
    rows = _rows(args.csv)
    head, units = rows[0], rows[1]
    col = {n: i for i, n in enumerate(head)}
    if "dram__bytes_read.sum" not in col:
        raise SystemExit("%s is not a `--page raw --csv` export of a `--set full` capture (no dram__bytes_read.sum); columns: %s"
                         % (args.csv, ", ".join(head[:40])))
    peak, peak_src = measured_hbm_gbs()

    def val(r, name, table):
        i = col[name]
        v = _num(r[i])
        return None if v is None else v * table.get(units[i], 1.0)

    extra = []
    for title, names, fmt in WANTED:
        for n in names:
            if n in col:
                extra.append((title, n, fmt))
                break
    L = ["# %s -- `ncu --set full` capture" % args.label, "", "Command (under gpurun, after the same command exited 0 without ncu):", "",
         "    " + args.command, "",
         "Read with `ncu -i <rep> --page raw --csv` and tabulated by `python -m paper_2602_17938_b200.ncu_summary full`.",
         "GB/s = (dram__bytes_read.sum + dram__bytes_write.sum) / gpu__time_duration.sum per launch; `of measured` is against",
         "%.1f GB/s (%s), `of ~8 TB/s` against the nominal figure BASELINE.json's north_star quotes." % (peak, peak_src), "",
         "| # | kernel | us | dram rd MB | dram wr MB | GB/s | of measured | of ~8 TB/s | " + " | ".join(t for t, _, _ in extra) + " |",
         "|---|---|---|---|---|---|---|---|" + "---|" * len(extra)]
    traffic = None
    n = 0
    for r in rows[2:]:
        if len(r) <= col["dram__bytes_read.sum"] or _num(r[col["gpu__time_duration.sum"]]) is None:
            continue
        k = short_name(r[col["Kernel Name"]])
        t = val(r, "gpu__time_duration.sum", UNIT_SECONDS)
        rd, wr = val(r, "dram__bytes_read.sum", UNIT_BYTES), val(r, "dram__bytes_write.sum", UNIT_BYTES)
        gbs = (rd + wr) / t / 1e9
        cells = []
        for _, name, fmt in extra:
            v = _num(r[col[name]])
            cells.append("-" if v is None else fmt % v)
        L.append("| %d | %s | %.1f | %.1f | %.1f | %.0f | %.3f | %.3f | %s |" % (n, k, t * 1e6, rd / 1e6, wr / 1e6, gbs, gbs / peak,
                                                                                 gbs / NOMINAL_HBM_GBS, " | ".join(cells)))
        if traffic is None and args.traffic_kernel and args.traffic_kernel in k:
            traffic = dict(bytes=int(round(rd + wr)), read=int(round(rd)), written=int(round(wr)), kernel=k, launch=n,
                           us=round(t * 1e6, 2), source=os.path.relpath(args.out, ROOT))
        n += 1
    if args.note:
        L += ["", args.note]
    open(args.out, "w").write("\n".join(L) + "\n")
    print("wrote", args.out, "(%d launches)" % n)
    if args.traffic:
        if traffic is None:
            raise SystemExit("no launch of a kernel named *%s* in the capture" % args.traffic_kernel)
        d = json.load(open(args.traffic)) if os.path.exists(args.traffic) else {}
        d[args.traffic_key] = traffic
        json.dump(d, open(args.traffic, "w"), indent=1, sort_keys=True)
        open(args.traffic, "a").write("\n")
        print("traffic[%s] = %d bytes -> %s" % (args.traffic_key, traffic["bytes"], args.traffic))


def main(argv=None):
    ap = argparse.ArgumentParser(description=__doc__.split("\n")[0])
    sub = ap.add_subparsers(dest="what", required=True)
    a = sub.add_parser("launches")
    a.add_argument("csv")
    a.add_argument("--out", required=True)
    a.add_argument("--command", required=True)
    a.add_argument("--label", default="r03")
    a.add_argument("--frame-launches", type=int, default=16, help="launches of one frame to list one by one (0: none)")
    a.add_argument("--frame-start", type=int, default=32, help="index (among the library's launches) of that frame's first launch")
    a.add_argument("--head", type=int, default=0, help="tabulate the first N library launches separately (0: all in one table)")
    a.add_argument("--head-what", default="the timed frames")
    a.add_argument("--rest-what", default="other legs of the command")
    a.set_defaults(fn=launches)
    b = sub.add_parser("full")
    b.add_argument("csv")
    b.add_argument("--out", required=True)
    b.add_argument("--command", required=True)
    b.add_argument("--label", default="r03")
    b.add_argument("--note", default="")
    b.add_argument("--traffic", default="", help="JSON file to update with the dram bytes of --traffic-kernel's first launch")
    b.add_argument("--traffic-key", default="noise_S")
    b.add_argument("--traffic-kernel", default="k_noise_S_tma")
    b.set_defaults(fn=full)
    args = ap.parse_args(argv)
    args.fn(args)
    return 0


if __name__ == "__main__":
    sys.exit(main())
