"""Reduces Nsight Compute CSV exports to the markdown tables under profiles/ (so that the tables are reproducible from
tracked code).  No GPU needed.

  python -m paper_2607_03012_b200.profile_tables launches <launches.csv>
      <launches.csv> = the log of  ncu --metrics gpu__time_duration.sum --clock-control none --csv --log-file <launches.csv> <cmd>
      -> per kernel: launches, total and mean duration, share of the listed GPU time

  python -m paper_2607_03012_b200.profile_tables full <raw.csv> [kernel-regex]
      <raw.csv> = ncu -i <report.ncu-rep> --page raw --csv   of an  ncu --set full --clock-control none  capture
      -> per captured kernel (first launch of each name): duration, DRAM bytes read / written and throughput, tensor-pipe,
         issue-slot, L2 figures, registers

  python -m paper_2607_03012_b200.profile_tables reduce <raw.csv>
      -> the same columns of every captured launch as a small CSV (kernel name, units row): the form committed under profiles/
         (bench.py reads roofline.traffic from it); `full` accepts it as well
"""
from __future__ import annotations

import collections
import csv
import io
import re
import sys

_UNIT = {"ns": 1e-6, "us": 1e-3, "usecond": 1e-3, "ms": 1.0, "msecond": 1.0, "s": 1e3, "second": 1e3, "nsecond": 1e-6}
_BYTES = {"byte": 1.0, "Kbyte": 1e3, "Mbyte": 1e6, "Gbyte": 1e9, "Tbyte": 1e12}


def _short(name: str) -> str:
    m = re.search(r"(hva_\w+)(<[^>(]*>)?", name)
    if m:
        return m.group(1) + (m.group(2) or "")
    return re.sub(r"\(.*", "", name)[:70]


def _rows(path):
    lines = [l for l in open(path, errors="replace") if l.startswith('"')]
    return list(csv.reader(io.StringIO("".join(lines))))


def launches(path: str) -> str:
    rows = _rows(path)
    hdr = rows[0]
    kn, mn, mu, mv = hdr.index("Kernel Name"), hdr.index("Metric Name"), hdr.index("Metric Unit"), hdr.index("Metric Value")
    tot, cnt = collections.OrderedDict(), collections.Counter()
    for r in rows[1:]:
        if len(r) <= mv or r[mn] != "gpu__time_duration.sum":
            continue
        k = _short(r[kn])
        v = float(r[mv].replace(",", "")) * _UNIT.get(r[mu], 1e-6)
        tot[k] = tot.get(k, 0.0) + v
        cnt[k] += 1
    total = sum(tot.values())
    out = ["| kernel | launches | total ms | mean us | share |", "|---|---:|---:|---:|---:|"]
    for k, v in sorted(tot.items(), key=lambda kv: -kv[1]):
        out.append(f"| `{k}` | {cnt[k]} | {v:.3f} | {1e3 * v / cnt[k]:.1f} | {100 * v / total:.1f} % |")
    out.append(f"| all listed launches | {sum(cnt.values())} | {total:.3f} | | 100 % |")
    return "\n".join(out)


# column title -> (candidate metric names, kind)
_FULL = [("time ms", ["gpu__time_duration.sum"], "t"), ("DRAM rd GB", ["dram__bytes_read.sum"], "b"), ("DRAM wr GB", ["dram__bytes_write.sum"], "b"),
         ("DRAM %", ["dram__throughput.avg.pct_of_peak_sustained_elapsed"], "p"),
         ("tensor %", ["sm__pipe_tensor_subpipe_hmma_cycles_active.avg.pct_of_peak_sustained_active",
                       "sm__pipe_tensor_op_hmma_cycles_active.avg.pct_of_peak_sustained_active",
                       "sm__inst_executed_pipe_tensor.avg.pct_of_peak_sustained_active"], "p"),
         ("issue %", ["smsp__issue_active.avg.pct_of_peak_sustained_active", "sm__inst_issued.avg.pct_of_peak_sustained_active"], "p"),
         ("fp64 %", ["sm__pipe_fp64_cycles_active.avg.pct_of_peak_sustained_active"], "p"),
         ("warps %", ["sm__warps_active.avg.pct_of_peak_sustained_active"], "p"), ("L2 hit %", ["lts__t_sector_hit_rate.pct"], "p"),
         ("L2 thr %", ["lts__throughput.avg.pct_of_peak_sustained_elapsed"], "p"),
         ("warp inst M", ["smsp__inst_executed.sum", "sm__inst_executed.sum"], "m"), ("regs", ["launch__registers_per_thread"], "i")]


def _table(path):
    rows = list(csv.reader(open(path, errors="replace")))
    h = next(i for i, r in enumerate(rows) if "Kernel Name" in r)
    return rows[h], rows[h + 1], rows[h + 2:]


def _pick(hdr):
    cols = []
    for title, names, kind in _FULL:
        for m in names:
            if m in hdr:
                cols.append((hdr.index(m), title, kind, m))
                break
    return cols


def full(path: str, pattern: str = ".") -> str:
    hdr, units, rows = _table(path)
    kn = hdr.index("Kernel Name")
    cols = _pick(hdr)
    out = ["| kernel | " + " | ".join(t for _, t, _, _ in cols) + " |", "|---|" + "---:|" * len(cols)]
    seen = set()
    for r in rows:
        if len(r) <= kn:
            continue
        k = _short(r[kn])
        if k in seen or not re.search(pattern, k):
            continue
        seen.add(k)
        cells = []
        for i, _, kind, _ in cols:
            try:
                v = float(r[i].replace(",", ""))
            except ValueError:
                cells.append("n/a")
                continue
            if kind == "t":
                cells.append(f"{v * _UNIT.get(units[i], 1e-6):.4f}")
            elif kind == "b":
                cells.append(f"{v * _BYTES.get(units[i], 1.0) / 1e9:.4f}")
            elif kind == "m":
                cells.append(f"{v / 1e6:.2f}")
            elif kind == "i":
                cells.append(f"{int(v)}")
            else:
                cells.append(f"{v:.1f}")
        out.append(f"| `{k}` | " + " | ".join(cells) + " |")
    return "\n".join(out)


def reduce(path: str) -> str:
    """The columns above (plus the kernel name) of a raw export, as CSV with the units row: what is committed under profiles/."""
    hdr, units, rows = _table(path)
    kn = hdr.index("Kernel Name")
    cols = _pick(hdr)
    buf = io.StringIO()
    w = csv.writer(buf)
    w.writerow(["Kernel Name"] + [m for _, _, _, m in cols])
    w.writerow([""] + [units[i] for i, _, _, _ in cols])
    for r in rows:
        if len(r) > kn:
            w.writerow([r[kn]] + [r[i] for i, _, _, _ in cols])
    return buf.getvalue().rstrip("\n")


if __name__ == "__main__":
    if len(sys.argv) < 3 or sys.argv[1] not in ("launches", "full", "reduce"):
        raise SystemExit(__doc__)
    if sys.argv[1] == "launches":
        print(launches(sys.argv[2]))
    elif sys.argv[1] == "reduce":
        print(reduce(sys.argv[2]))
    else:
        print(full(sys.argv[2], sys.argv[3] if len(sys.argv) > 3 else "."))
