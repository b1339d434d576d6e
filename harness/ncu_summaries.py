"""Turns the CSV pages of Nsight Compute into the small text summaries kept under profiles/ (evidence tooling, not part
of the product path). Reads a file, writes CSV to stdout; nothing here runs a GPU.

  python -m harness.ncu_summaries launches RAW.csv
      RAW.csv = the log of `ncu --metrics gpu__time_duration.sum --clock-control none --csv --log-file RAW.csv <cmd>`
      -> id,kernel,block,grid,gpu__time_duration_ns (one line per launch) and, per kernel, its share of the total
  python -m harness.ncu_summaries opcodes SOURCE.csv [CELL_UPDATES]
      SOURCE.csv = `ncu -i X.ncu-rep --page source --csv --print-source sass`
      -> per SASS opcode: static count, executed warp instructions, executed thread instructions, shared-memory
         wavefronts (total and in excess of the ideal), stall samples; with CELL_UPDATES (the cell-updates of the captured
         launch) also thread instructions per cell-update, the unit the roofline discussion of DESIGN.md section 6 uses
  python -m harness.ncu_summaries metrics RAW_PAGE.csv [REGEX]
      RAW_PAGE.csv = `ncu -i X.ncu-rep --page raw --csv` -> metric,unit,value for the first captured kernel, keeping the
      metrics whose name matches REGEX (default: the counters the roofline discussion uses)
"""
import csv
import re
import sys
from collections import OrderedDict


def _rows(path):
    with open(path, newline="") as f:
        return [r for r in csv.reader(l for l in f if not l.startswith("=="))]


def launches(path, out=sys.stdout):
    rows = _rows(path)
    head = rows[0]
    col = {n: head.index(n) for n in ("ID", "Kernel Name", "Block Size", "Grid Size", "Metric Name", "Metric Value")}
    w = csv.writer(out)
    w.writerow(["id", "kernel", "block", "grid", "gpu__time_duration_ns"])
    per = OrderedDict()
    for r in rows[1:]:
        if len(r) <= col["Metric Value"] or r[col["Metric Name"]] != "gpu__time_duration.sum":
            continue
        name = re.sub(r"^void\s+", "", r[col["Kernel Name"]])
        name = re.sub(r"\(.*$", "", name).replace("gh::", "")
        ns = int(float(r[col["Metric Value"]].replace(",", "")))
        w.writerow([int(r[col["ID"]]) + 1, name, r[col["Block Size"]], r[col["Grid Size"]], ns])
        n, t = per.get(name, (0, 0))
        per[name] = (n + 1, t + ns)
    total = sum(t for _, t in per.values()) or 1
    w.writerow([])
    w.writerow(["kernel", "launches", "total_ns", "mean_ns", "share_of_all_kernel_time"])
    for name, (n, t) in per.items():
        w.writerow([name, n, t, round(t / n), "%.4f" % (t / total)])


def _opcode(source):
    s = source.strip()
    s = re.sub(r"^@!?U?P\d+\s+", "", s)          # predicate
    return s.split()[0].rstrip(";") if s else ""


def opcodes(path, cell_updates=None, out=sys.stdout):
    rows = _rows(path)
    hi = next(i for i, r in enumerate(rows) if "Source" in r and "Instructions Executed" in r)
    head = rows[hi]
    c = {n: head.index(n) for n in ("Source", "# Samples", "Instructions Executed", "Thread Instructions Executed",
                                    "L1 Wavefronts Shared", "L1 Wavefronts Shared Excessive")}
    num = lambda r, n: int(float(r[c[n]].replace(",", "") or 0)) if r[c[n]] not in ("-", "") else 0
    agg = {}
    for r in rows[hi + 1:]:
        if len(r) != len(head):
            continue
        full = _opcode(r[c["Source"]])
        if not full:
            continue
        for key in {full.split(".")[0], full}:
            a = agg.setdefault(key, [0, 0, 0, 0, 0, 0])
            a[0] += 1
            a[1] += num(r, "Instructions Executed")
            a[2] += num(r, "Thread Instructions Executed")
            a[3] += num(r, "L1 Wavefronts Shared")
            a[4] += num(r, "L1 Wavefronts Shared Excessive")
            a[5] += num(r, "# Samples")
    base = {k: v for k, v in agg.items() if "." not in k}
    tot = [sum(v[i] for v in base.values()) for i in range(6)]
    w = csv.writer(out)
    cols = ["opcode", "static_count", "warp_instr_executed", "thread_instr_executed", "share_of_warp_instr",
            "smem_wavefronts", "smem_wavefronts_excess", "stall_samples"]
    if cell_updates:
        cols.append("thread_instr_per_cell_update")
    w.writerow(cols)

    def line(k, v):
        r = [k, v[0], v[1], v[2], "%.4f" % (v[1] / max(tot[1], 1)), v[3], v[4], v[5]]
        if cell_updates:
            r.append("%.2f" % (v[2] / cell_updates))
        w.writerow(r)

    line("ALL", tot)
    w.writerow(["# by base opcode"])
    for k, v in sorted(base.items(), key=lambda kv: -kv[1][1]):
        line(k, v)
    w.writerow(["# by full mnemonic (modifiers kept), executed at least once"])
    for k, v in sorted(((k, v) for k, v in agg.items() if "." in k and v[1] > 0), key=lambda kv: -kv[1][1]):
        line(k, v)


DEFAULT_METRICS = (r"^(gpu__time_duration|launch__(grid_size|block_size|registers_per_thread|occupancy_limit|waves)|"
                   r"dram__bytes_(read|write)\.sum$|dram__throughput|sm__throughput|smsp__issue_active|smsp__inst_executed\.|"
                   r"smsp__thread_inst_executed\.sum|sm__inst_executed_pipe_(fma|alu|fmaheavy|fmalite|xu|lsu|uniform)|"
                   r"sm__pipe_(fma|alu|fmaheavy|xu)_cycles_active|smsp__warps_(active|eligible)|smsp__issue_inst0|"
                   r"smsp__average_warp.*issue_stalled.*_per_warp_active|smsp__average_warps_issue_stalled.*ratio|"
                   r"l1tex__data_pipe_lsu_wavefronts|l1tex__data_bank_conflicts_pipe_lsu|smsp__sass_l1tex_data_bank|"
                   r"sm__warps_active|sm__cycles_(active|elapsed)\.(avg|max)$|smsp__cycles_active\.avg$|lts__t_sector_hit_rate)")


def metrics(path, regex=DEFAULT_METRICS, out=sys.stdout):
    rows = _rows(path)
    head, units, vals = rows[0], rows[1], rows[2]
    w = csv.writer(out)
    w.writerow(["metric", "unit", "value"])
    w.writerow(["kernel", "", vals[head.index("Kernel Name")]])
    rx = re.compile(regex)
    for name, u, v in zip(head, units, vals):
        short = name.split(".", 2)[-1] if name.count(".") >= 2 and name.split(".")[1] == "TriageCompute" else name
        if rx.search(short):
            w.writerow([short, u, v])


if __name__ == "__main__":
    if len(sys.argv) >= 3 and sys.argv[1] == "metrics":
        metrics(sys.argv[2], sys.argv[3] if len(sys.argv) > 3 else DEFAULT_METRICS)
        sys.exit(0)
    if len(sys.argv) >= 3 and sys.argv[1] == "launches":
        launches(sys.argv[2])
    elif len(sys.argv) >= 3 and sys.argv[1] == "opcodes":
        opcodes(sys.argv[2], float(sys.argv[3]) if len(sys.argv) > 3 else None)
    else:
        sys.exit(__doc__)
