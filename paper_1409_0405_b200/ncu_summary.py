"""Summarise an Nsight Compute capture of one right-hand side as text (what `profiles/` keeps and `bench.py` reads for
`roofline.traffic`).

  python -m paper_1409_0405_b200.ncu_summary REPORT.ncu-rep --bench BENCH.json --prec f64 [--csv OUT.csv] [--append]
  python -m paper_1409_0405_b200.ncu_summary --launches LAUNCHES.csv      (markdown table of an ncu launch list)

REPORT.ncu-rep: `ncu --set full` capture of the first launches of bench.py's timed region (one right-hand side = every kernel from
S1 to the last fused divergence kernel; the command is recorded in the .md next to the CSV).  BENCH.json: the line
`python bench.py --kernels` printed, which names the steps in launch order (`kernels_f64` / `kernels_f32`).  The boundary-condition
launches are folded into their step (S2: k_con_u + k_bc_con_u, S7: k_comm_flux + k_bc_comm_flux), so launches map one-to-one to
the steps of `fr_profile_stage_kernels`.  Columns of the CSV: precision, step, DRAM bytes (read + write), duration ms, registers
per thread, dynamic shared memory bytes, FP64-tensor / FMA pipe utilisation %, kernel name.  Needs `ncu` on PATH (no GPU).
"""
import argparse
import csv
import io
import json
import re
import subprocess
import sys


def read_raw(report):
    out = subprocess.run(["ncu", "-i", report, "--page", "raw", "--csv"], capture_output=True, text=True, check=True).stdout
    rows = list(csv.reader(io.StringIO(out)))
    hdr, units, data = rows[0], rows[1], rows[2:]
    return hdr, units, data


def to_bytes(value, unit):
    v = float(value.replace(",", ""))
    return v * {"byte": 1.0, "Kbyte": 1e3, "Mbyte": 1e6, "Gbyte": 1e9, "Tbyte": 1e12}.get(unit, 1.0)


def to_ms(value, unit):
    v = float(value.replace(",", ""))
    return v * {"ns": 1e-6, "us": 1e-3, "ms": 1.0, "s": 1e3}.get(unit, 1.0)


def launch_table(path):
    """Markdown table of an `ncu --metrics gpu__time_duration.sum --csv` launch list: launches, total and mean time, share per kernel."""
    lines = [l for l in open(path) if l.startswith('"')]
    rows = list(csv.reader(io.StringIO("".join(lines))))
    col = {h: i for i, h in enumerate(rows[0])}
    agg = {}
    for r in rows[1:]:
        if r[col["Metric Name"]] != "gpu__time_duration.sum":
            continue
        name = re.sub(r"\(.*", "", r[col["Kernel Name"]]).split("::")[-1].replace("void ", "")
        key = "`%s` x%s" % (name, r[col["Block Size"]].strip("()").split(",")[0])
        ms = to_ms(r[col["Metric Value"]], r[col["Metric Unit"]])
        a = agg.setdefault(key, [0, 0.0])
        a[0] += 1
        a[1] += ms
    tot = sum(a[1] for a in agg.values())
    out = ["| kernel x threads per CTA | launches | total ms | share | mean ms |", "|---|---|---|---|---|"]
    for k, (n, ms) in sorted(agg.items(), key=lambda kv: -kv[1][1]):
        out.append("| %s | %d | %.3f | %.1f %% | %.3f |" % (k, n, ms, 100 * ms / tot, ms / n))
    out.append("| total | %d | %.3f | | |" % (sum(a[0] for a in agg.values()), tot))
    return "\n".join(out)


def main():
    if len(sys.argv) == 3 and sys.argv[1] == "--launches":
        print(launch_table(sys.argv[2]))
        return
    ap = argparse.ArgumentParser()
    ap.add_argument("report")
    ap.add_argument("--bench", required=True)
    ap.add_argument("--prec", default="f64", choices=["f64", "f32"])
    ap.add_argument("--csv", default=None)
    ap.add_argument("--append", action="store_true")
    args = ap.parse_args()
    names = None
    for line in open(args.bench):
        if line.startswith("{"):
            d = json.loads(line)
            names = [k["name"] for k in d["kernels_" + args.prec]]
    if not names:
        raise SystemExit("no kernels_%s in %s (run bench.py with --kernels)" % (args.prec, args.bench))
    hdr, units, data = read_raw(args.report)
    col = {h: i for i, h in enumerate(hdr)}

    def get(r, k):
        return r[col[k]] if k in col else ""

    steps = []
    for r in data:
        kn = get(r, "Kernel Name")
        short = re.sub(r"\(.*", "", kn).split("::")[-1]
        cls = "S2" if "con_u" in kn else ("S7" if "comm_flux" in kn else None)
        rec = dict(kernel=short,
                   dram=to_bytes(get(r, "dram__bytes_read.sum"), units[col["dram__bytes_read.sum"]]) +
                   to_bytes(get(r, "dram__bytes_write.sum"), units[col["dram__bytes_write.sum"]]),
                   ms=to_ms(get(r, "gpu__time_duration.sum"), units[col["gpu__time_duration.sum"]]),
                   regs=get(r, "launch__registers_per_thread"), smem=get(r, "launch__shared_mem_per_block_dynamic"),
                   dmma=get(r, "sm__pipe_tensor_subpipe_dmma_cycles_active.avg.pct_of_peak_sustained_active"),
                   fma=get(r, "sm__pipe_fma_cycles_active.avg.pct_of_peak_sustained_active"), cls=cls)
        if cls and steps and steps[-1]["cls"] == cls:
            steps[-1]["dram"] += rec["dram"]
            steps[-1]["ms"] += rec["ms"]
        else:
            steps.append(rec)
        if len(steps) > len(names):
            break
    steps = steps[:len(names)]
    if len(steps) != len(names):
        raise SystemExit("capture holds %d steps, bench names %d: capture at least one whole right-hand side" % (len(steps), len(names)))
    f = open(args.csv, "a" if args.append else "w") if args.csv else sys.stdout
    for n, s in zip(names, steps):
        f.write("%s,%s,%.0f,%.4f,%s,%s,%s,%s,%s\n" % (args.prec, n, s["dram"], s["ms"], s["regs"], s["smem"], s["dmma"], s["fma"], s["kernel"]))
    if args.csv:
        f.close()


if __name__ == "__main__":
    main()
