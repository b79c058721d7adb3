"""Turns Nsight Compute exports of a bench.py run into the text kept under profiles/.

    python -m paper_2607_04206_b200.ncu_summary launches NAME=launches.csv [NAME=...]
        per-kernel launch count / mean / min / max / share from `ncu --metrics gpu__time_duration.sum --csv` launch lists
    python -m paper_2607_04206_b200.ncu_summary full NAME=raw.csv [NAME=...] [--traffic profiles/traffic.json]
        the roofline-relevant metrics of the first kernel in each `ncu -i X.ncu-rep --page raw --csv` export; with --traffic
        also writes {"sources_hash": <csrc hash>, "workloads": {NAME: dram bytes read + written}} for bench.py's `traffic`

It only reads CSV text and prints markdown: no GPU, no CUDA extension needed.
"""
from __future__ import annotations

import csv
import json
import re
import sys

FULL_METRICS = [
    ("gpu__time_duration.sum", "gpu__time_duration.sum"),
    ("dram__bytes_read.sum", "dram__bytes_read.sum"),
    ("dram__bytes_write.sum", "dram__bytes_write.sum"),
    ("gpu__dram_throughput.avg.pct_of_peak_sustained_elapsed", "gpu__dram_throughput % of peak"),
    ("sm__pipe_tensor_cycles_active.avg.pct_of_peak_sustained_active", "sm__pipe_tensor_cycles_active % of peak (active)"),
    ("sm__inst_executed_pipe_xu.avg.pct_of_peak_sustained_active", "sm__inst_executed_pipe_xu % of peak (MUFU)"),
    ("sm__inst_executed_pipe_fma.avg.pct_of_peak_sustained_active", "sm__inst_executed_pipe_fma % of peak"),
    ("sm__inst_executed_pipe_alu.avg.pct_of_peak_sustained_active", "sm__inst_executed_pipe_alu % of peak"),
    ("smsp__issue_active.avg.pct_of_peak_sustained_active", "smsp__issue_active % of peak"),
    ("lts__t_sector_hit_rate.pct", "lts__t_sector_hit_rate"),
    ("smsp__inst_executed.sum", "smsp__inst_executed.sum"),
    ("launch__registers_per_thread", "launch__registers_per_thread"),
    ("launch__grid_size", "launch__grid_size"),
    ("launch__block_size", "launch__block_size"),
    ("launch__occupancy_limit_shared_mem", "launch__occupancy_limit_shared_mem (CTAs/SM)"),
]


def short_kernel(name: str) -> str:
    name = re.sub(r"\(CUtensorMap_st.*$", "", name)
    name = re.sub(r"^void ", "", name)
    name = name.replace("(int)", "").replace("(bool)", "")
    return name.split("(")[0].strip()


def to_bytes(value: float, unit: str) -> float:
    scale = {"byte": 1.0, "Kbyte": 1e3, "Mbyte": 1e6, "Gbyte": 1e9, "Tbyte": 1e12}
    return value * scale.get(unit, 1.0)


def to_us(value: float, unit: str) -> float:
    scale = {"ns": 1e-3, "us": 1.0, "usecond": 1.0, "ms": 1e3, "msecond": 1e3, "nsecond": 1e-3, "s": 1e6, "second": 1e6}
    return value * scale.get(unit, 1.0)


def num(x: str) -> float:
    return float(x.replace(",", "")) if x not in ("", "n/a") else float("nan")


def launches(pairs):
    print("| workload | kernel | launches | mean ns | min ns | max ns | share |")
    print("|---|---|---|---|---|---|---|")
    for name, path in pairs:
        rows = [r for r in csv.reader(l for l in open(path) if not l.startswith("=="))]
        head = next(i for i, r in enumerate(rows) if "Kernel Name" in r)
        h = rows[head]
        ik, iv, iu, im = h.index("Kernel Name"), h.index("Metric Value"), h.index("Metric Unit"), h.index("Metric Name")
        per = {}
        for r in rows[head + 1:]:
            if len(r) <= iv or r[im] != "gpu__time_duration.sum":
                continue
            per.setdefault(short_kernel(r[ik]), []).append(to_us(num(r[iv]), r[iu]) * 1e3)
        ours = {k: v for k, v in per.items() if not k.startswith("at::") and "at::native" not in k}
        total = sum(sum(v) for v in ours.values())
        for k, v in sorted(ours.items(), key=lambda kv: -sum(kv[1])):
            print(f"| {name} | {k} | {len(v)} | {sum(v) / len(v):,.0f} | {min(v):,.0f} | {max(v):,.0f} | {100 * sum(v) / total:.1f} % |")


def full(pairs, traffic_path):
    cols, tables = [], []
    traffic = {}
    for name, path in pairs:
        rows = list(csv.reader(open(path)))
        h, units, first = rows[0], rows[1], rows[2]
        d = {k: (first[i], units[i]) for i, k in enumerate(h)}
        kern = short_kernel(d["Kernel Name"][0])
        cols.append(f"{name}: {kern}")
        tables.append(d)
        rd = to_bytes(num(d["dram__bytes_read.sum"][0]), d["dram__bytes_read.sum"][1])
        wr = to_bytes(num(d["dram__bytes_write.sum"][0]), d["dram__bytes_write.sum"][1])
        traffic[name] = rd + wr
    print("| metric | " + " | ".join(cols) + " |")
    print("|---|" + "---|" * len(cols))
    for key, label in FULL_METRICS:
        cells = []
        for d in tables:
            v, u = d.get(key, ("", ""))
            cells.append(f"{v} {u}".strip() if v != "" else "n/a")
        print(f"| {label} | " + " | ".join(cells) + " |")
    print("| traffic (read + write), bytes | " + " | ".join(f"{traffic[n]:,.0f}" for n, _ in pairs) + " |")
    if traffic_path:
        from .build import sources_hash
        with open(traffic_path, "w") as f:
            json.dump({"sources_hash": sources_hash(), "workloads": traffic,
                       "_source": "ncu --set full, dram__bytes_read.sum + dram__bytes_write.sum of the attention kernel, first captured "
                                  "launch; written by python -m paper_2607_04206_b200.ncu_summary full ... --traffic"}, f, indent=1)
            f.write("\n")


def main(argv):
    if len(argv) < 2 or argv[0] not in ("launches", "full"):
        print(__doc__)
        return 2
    traffic_path = None
    if "--traffic" in argv:
        i = argv.index("--traffic")
        traffic_path = argv[i + 1]
        argv = argv[:i] + argv[i + 2:]
    pairs = [a.split("=", 1) for a in argv[1:]]
    if argv[0] == "launches":
        launches(pairs)
    else:
        full(pairs, traffic_path)
    return 0


if __name__ == "__main__":
    sys.exit(main(sys.argv[1:]))
