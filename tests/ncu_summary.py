"""Turns the ncu exports kept under profiles/ into the tables of the profile summaries (not a test; nothing here runs on
a GPU).

    python tests/ncu_summary.py launches profiles/r02_mg_launches.csv [--first N --last M]
        per-kernel count, total and mean gpu__time_duration and share, from an
        `ncu --metrics gpu__time_duration.sum --csv` launch list
    python tests/ncu_summary.py raw <file>.csv [metric ...]
        one row per metric, one column per launch, from `ncu -i <rep> --page raw --csv`
"""
import csv
import re
import sys
from collections import OrderedDict

RAW_DEFAULT = [
    "gpu__time_duration.sum", "dram__bytes_read.sum", "dram__bytes_write.sum", "launch__registers_per_thread",
    "launch__block_size", "launch__grid_size", "sm__warps_active.avg.pct_of_peak_sustained_active",
    "lts__t_sector_hit_rate.pct", "smsp__inst_executed.sum",
    "smsp__average_warps_issue_stalled_long_scoreboard_per_issue_active.ratio",
    "smsp__average_warps_issue_stalled_short_scoreboard_per_issue_active.ratio",
    "smsp__average_warps_issue_stalled_barrier_per_issue_active.ratio",
    "smsp__average_warps_issue_stalled_wait_per_issue_active.ratio",
    "l1tex__data_pipe_lsu_wavefronts_mem_shared.sum", "l1tex__data_bank_conflicts_pipe_lsu_mem_shared.sum",
]


def short_name(name):
    name = re.sub(r"\(anonymous namespace\)::|<unnamed>::|ifl::|void ", "", name)
    name = re.sub(r"\(.*$", "", name)
    return name.replace("(int)", "").replace("(bool)", "")


def read_ncu_csv(path):
    rows = list(csv.reader(line for line in open(path) if not line.startswith("==")))
    start = next(i for i, r in enumerate(rows) if "Kernel Name" in r)
    return rows[start], rows[start + 1:]


def launches(path, first=None, last=None):
    hdr, data = read_ncu_csv(path)
    i_name, i_val = hdr.index("Kernel Name"), hdr.index("Metric Value")
    i_unit, i_metric = hdr.index("Metric Unit"), hdr.index("Metric Name")
    i_grid = hdr.index("Grid Size") if "Grid Size" in hdr else None
    per = OrderedDict()
    items = [r for r in data if len(r) > i_val and r[i_metric] == "gpu__time_duration.sum"]
    items = items[first or 0:last]
    for r in items:
        t = float(r[i_val].replace(",", ""))
        t *= {"ns": 1e-3, "us": 1.0, "ms": 1e3, "s": 1e6}.get(r[i_unit], 1.0)
        key = (short_name(r[i_name]), r[i_grid] if i_grid is not None else "")
        n, tot = per.get(key, (0, 0.0))
        per[key] = (n + 1, tot + t)
    total = sum(t for _, t in per.values())
    print(f"{len(items)} launches, {total / 1e3:.2f} ms")
    print(f"{'kernel':<44}{'grid':>16}{'n':>6}{'total us':>12}{'mean us':>10}{'share':>8}")
    for (name, grid), (n, tot) in sorted(per.items(), key=lambda kv: -kv[1][1]):
        print(f"{name:<44}{grid:>16}{n:>6}{tot:>12.1f}{tot / n:>10.1f}{100 * tot / total:>7.1f}%")


def raw(path, metrics):
    hdr, data = read_ncu_csv(path)
    units, data = data[0], data[1:]
    idx = {h: i for i, h in enumerate(hdr)}
    print("| metric | unit | " + " | ".join(short_name(d[idx["Kernel Name"]]) for d in data) + " |")
    print("|---|---|" + "---|" * len(data))
    for m in metrics or RAW_DEFAULT:
        if m in idx:
            vals = []
            for d in data:
                try:
                    vals.append(f"{float(d[idx[m]].replace(',', '')):.4g}")
                except ValueError:
                    vals.append(d[idx[m]])
            print(f"| {m} | {units[idx[m]]} | " + " | ".join(vals) + " |")


if __name__ == "__main__":
    if len(sys.argv) >= 3 and sys.argv[1] == "launches":
        a = sys.argv[3:]
        first = int(a[a.index("--first") + 1]) if "--first" in a else None
        last = int(a[a.index("--last") + 1]) if "--last" in a else None
        launches(sys.argv[2], first, last)
    elif len(sys.argv) >= 3 and sys.argv[1] == "raw":
        raw(sys.argv[2], sys.argv[3:])
    else:
        print(__doc__)
