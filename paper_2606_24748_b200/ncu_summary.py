"""Turn an `ncu --set full` capture into the text evidence kept under profiles/.

    ncu -i gpurun_out/prof.ncu-rep --page raw --csv > gpurun_out/prof_raw.csv
    python -m paper_2606_24748_b200.ncu_summary gpurun_out/prof_raw.csv [more_raw.csv ...] \
        --traffic profiles/ncu_traffic.csv --table profiles/<name>.md

Reads the raw-page CSV (one row per profiled launch, a units row under the header), averages the launches of each
kernel and writes (a) `--traffic`: bench.py's kernel name, dram__bytes_read.sum + dram__bytes_write.sum per launch
(what bench.py reports as roofline.traffic) and (b) `--table`: a markdown table of the counters DESIGN.md quotes.
Nothing here runs on the GPU or touches the hot path."""
from __future__ import annotations

import argparse
import csv
import sys
from collections import OrderedDict

# substring of the demangled kernel name -> the name bench.py uses
BENCH_NAMES = [
    ("spmv_flat_kernel<3, 6", "spmv_P"), ("spmv_kernel<3, 3", "spmv_A"), ("spmv_kernel<6, 3", "spmv_Pt"),
    ("stream_product_kernel<3, 3, 6, 256, 0, 0", "ptap_stage1_AP"), ("stream_product_kernel<6, 3, 6", "ptap_stage2_RAP"),
    ("stream_product_kernel<3, 3, 6, 256, 0, 1", "prolongator_smooth"), ("bcoo_flat_kernel<9", "bcoo_set_values"),
    ("bcoo_sum_kernel<9", "bcoo_set_values_per_value"),
    ("spmv_kernel<6, 6", "spmv_6x6"), ("cheb_update_kernel", "cheb_update"), ("trigemv_kernel", "trigemv"),
]
METRICS = OrderedDict([
    ("gpu__time_duration.sum", "duration"), ("dram__bytes_read.sum", "DRAM read"), ("dram__bytes_write.sum", "DRAM write"),
    ("gpu__dram_throughput.avg.pct_of_peak_sustained_elapsed", "DRAM % of ncu peak"),
    ("launch__registers_per_thread", "registers / thread"), ("sm__warps_active.avg.pct_of_peak_sustained_active", "warps active %"),
    ("sm__pipe_fp64_cycles_active.avg.pct_of_peak_sustained_active", "fp64 pipe active %"),
    ("l1tex__data_pipe_lsu_wavefronts_mem_shared.sum", "shared-memory wavefronts"),
    ("smsp__inst_executed_op_shared_ld.sum", "LDS instructions"),
])
SCALE = {"byte": 1.0, "Kbyte": 1e3, "Mbyte": 1e6, "Gbyte": 1e9, "Tbyte": 1e12, "nsecond": 1e-9, "usecond": 1e-6,
         "msecond": 1e-3, "second": 1.0, "ns": 1e-9, "us": 1e-6, "ms": 1e-3, "s": 1.0}


def bench_name(kernel: str) -> str | None:
    flat = kernel.replace("(bool)", "").replace("(int)", "").replace("(bsramg::Epilogue)", "")
    for sub, name in BENCH_NAMES:
        if sub in flat:
            return name
    return None


def load(path: str):
    rows = list(csv.reader(open(path, newline="")))
    start = next(i for i, r in enumerate(rows) if "Kernel Name" in r)
    head, units = rows[start], rows[start + 1]
    col = {h: i for i, h in enumerate(head)}
    out = OrderedDict()
    for r in rows[start + 2:]:
        if len(r) < len(head):
            continue
        k = r[col["Kernel Name"]]
        rec = out.setdefault(k, {m: [] for m in METRICS})
        for m in METRICS:
            if m in col and r[col[m]] not in ("", "n/a"):
                try:
                    rec[m].append(float(r[col[m]].replace(",", "")) * SCALE.get(units[col[m]], 1.0))
                except ValueError:
                    pass
    return out


def mean(v):
    return sum(v) / len(v) if v else None


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("raw_csv", nargs="+")
    ap.add_argument("--traffic", help="write bench.py's traffic table (profiles/ncu_traffic.csv)")
    ap.add_argument("--table", help="write a markdown table of the counters")
    ap.add_argument("--command", default="", help="the capture command, recorded in the table's header")
    a = ap.parse_args()
    data = OrderedDict()
    for path in a.raw_csv:
        for k, rec in load(path).items():
            tgt = data.setdefault(k, {m: [] for m in METRICS})
            for m in METRICS:
                tgt[m] += rec[m]
    if a.traffic:
        with open(a.traffic, "w") as f:
            f.write("kernel,dram_bytes_per_launch,launches,kernel_name\n")
            for k, rec in data.items():
                name, rd, wr = bench_name(k), mean(rec["dram__bytes_read.sum"]), mean(rec["dram__bytes_write.sum"])
                if name and rd is not None and wr is not None:
                    f.write(f"{name},{int(rd + wr)},{len(rec['dram__bytes_read.sum'])},\"{k[:100]}\"\n")
    lines = []
    if a.command:
        lines += ["Capture command (committed files only):", "", "```", a.command, "```", ""]
    lines += ["| kernel | launches | " + " | ".join(METRICS.values()) + " |", "|---|---|" + "---|" * len(METRICS)]
    for k, rec in data.items():
        cells = []
        for m in METRICS:
            v = mean(rec[m])
            if v is None:
                cells.append("-")
            elif m.startswith("gpu__time"):
                cells.append(f"{v * 1e3:.3f} ms")
            elif "bytes" in m:
                cells.append(f"{v / 1e9:.3f} GB")
            elif "wavefronts" in m or "inst_executed" in m:
                cells.append(f"{v / 1e6:.1f} M")
            else:
                cells.append(f"{v:.1f}")
        n = max(len(rec[m]) for m in METRICS)
        lines.append(f"| `{(bench_name(k) or '')} {k[:70]}` | {n} | " + " | ".join(cells) + " |")
    text = "\n".join(lines) + "\n"
    if a.table:
        open(a.table, "w").write(text)
    else:
        sys.stdout.write(text)


if __name__ == "__main__":
    main()
