"""Per-kernel roofline table of one right-hand side as markdown (what `profiles/r02_a_kernels.md` holds).

  python -m paper_1409_0405_b200.kernel_table BENCH.json [--traffic TRAFFIC.csv] [--prev PREV_BENCH.json] > table.md
  python -m paper_1409_0405_b200.kernel_table --gemm BENCH.json          (the `gemm` object of the line as a table)

BENCH.json: the line `python bench.py --kernels` printed (per-kernel CUDA-event times, algorithmic bytes and flops of
`fr_profile_stage_kernels`, the peaks measured in the same run, the plans `fr_setup` chose).  TRAFFIC.csv: the DRAM bytes and pipe
utilisation per kernel that `paper_1409_0405_b200.ncu_summary` extracts from an `ncu --set full` capture.  PREV_BENCH.json: an earlier
line whose times go in brackets.  `frac` = max(algorithmic GB/s / HBM peak, flops / pipe peak): the FP64 tensor pipe for FP64,
the FP32 FMA pipe for FP32.  No GPU needed.
"""
import argparse
import csv
import json
import sys


def load(path):
    for line in open(path):
        line = line.strip()
        if line.startswith("{") and '"metric"' in line:
            return json.loads(line)
    raise SystemExit("no bench line in %s" % path)


def gemm_table(d):
    """The `gemm` object of a bench line (operator product alone, eight shapes x two precisions) as a markdown table."""
    out = ["| shape | M x K | N | FP64 ms | GB/s | TF | bound | frac | library ms | FP32 ms | GB/s | TF | bound | frac | library ms |",
           "|" + "---|" * 15]
    rows = {}
    for g in d["gemm"]:
        rows.setdefault((g["shape"], g["M"], g["K"]), {})[g["dtype"]] = g
    for (shape, M, K), r in rows.items():
        cells = [shape, "%d x %d" % (M, K), "%d" % r["f64"]["N"]]
        for prec in ("f64", "f32"):
            g = r[prec]
            cells += ["%.3f" % g["ms"], "%.0f" % g["gbs"], "%.1f" % g["tflops"], g["bound"], "%.2f" % g["frac"], "%.3f" % g["library_gemm_ms"]]
        out.append("| " + " | ".join(cells) + " |")
    return "\n".join(out)


def single_table(d):
    """A line that carries one precision only (bench.py --workload config5): headline, per-kernel table, plan."""
    prec = d["dtype"]
    ks = d["kernels_" + prec]
    hbm = d["roofline"]["hbm"]["peak"]
    peak = d["peaks"]["fp64_tensor_tflops" if prec == "f64" else "fp32_ffma_tflops"]
    tot = sum(k["ms"] for k in ks)
    out = ["Workload: %s; %d DOF; %s; dt = %g." % (d["config"]["workload"], d["config"]["dof"], prec.upper(), d["config"]["dt"]), "",
           "* **%.3f GDOF-RHS/s** (%.1f ms per RK45 step, %d kernel launches in the timed region of %d steps). SM clock %.0f of %.0f MHz, reasons %s."
           % (d["value"], d["ms_per_step"], d["gpu_launches"], d["steps"], d["clocks"]["sm_mhz"], d["clocks"]["sm_max_mhz"], d["clocks"]["reasons"]),
           "* end to end through `fr_rk_step_host` (%.2f GB of pinned host state in, one step, %.2f GB out): %.3f GDOF-RHS/s."
           % (d["e2e"]["h2d_bytes_per_step"] / 1e9, d["e2e"]["d2h_bytes_per_step"] / 1e9, d["e2e"]["value"]),
           "* one right-hand side as an RK stage runs it (`fr_profile_stage_kernels`, CUDA events, mean of 3): operator products incl. fused point-wise "
           "work %.1f ms, stand-alone point-wise (S6) %.1f ms, interface kernels %.1f ms; total %.1f ms."
           % (d["kernel_groups"]["operator_products_incl_fused_pointwise_ms"], d["kernel_groups"]["pointwise_flux_ms"],
              d["kernel_groups"]["interface_ms"], d["kernel_groups"]["total_ms"]), "",
           "| kernel | ms | share | algorithmic GB/s | of %.0f GB/s | TFLOP/s | of %.1f |" % (hbm, peak), "|---|---|---|---|---|---|---|"]
    for k in ks:
        gbs, tf = k["alg_bytes"] / k["ms"] / 1e6, k["flops"] / k["ms"] / 1e9
        out.append("| %s | %.2f | %.1f %% | %.0f | %.0f %% | %.1f | %.0f %% |" % (k["name"], k["ms"], 100 * k["ms"] / tot, gbs, 100 * gbs / hbm, tf, 100 * tf / peak))
    out += ["", "Plan chosen by `fr_setup` (`fr_plan_describe`):", "", "```"] + list(d["plan"]) + ["```", ""]
    return "\n".join(out)


def main():
    if len(sys.argv) == 3 and sys.argv[1] == "--gemm":
        print(gemm_table(load(sys.argv[2])))
        return
    ap = argparse.ArgumentParser()
    ap.add_argument("bench")
    ap.add_argument("--traffic", default=None)
    ap.add_argument("--prev", default=None)
    args = ap.parse_args()
    d = load(args.bench)
    prev = load(args.prev) if args.prev else None
    traffic = {}
    if args.traffic:
        for r in csv.reader(open(args.traffic)):
            if len(r) >= 8:
                traffic[(r[0], r[1])] = dict(dram=float(r[2]), pipe64=float(r[6]), pipe32=float(r[7]))
    if "kernels_f64" not in d or "fp32" not in d:
        sys.stdout.write(single_table(d))
        return
    hbm = d["roofline"]["hbm"]["peak"]
    pk = d["peaks"]
    peak = {"f64": pk["fp64_tensor_tflops"], "f32": pk["fp32_ffma_tflops"]}
    out = []
    out.append("HBM peak %.1f GB/s (%s); FP64 tensor pipe %.2f TFLOP/s (`fr_probe_dmma`), FP32 FMA pipe %.2f TFLOP/s (`fr_probe_peaks`), "
               "both measured in the same run." % (hbm, d["roofline"]["hbm"]["peak_source"], peak["f64"], peak["f32"]))
    if "ffma2_tflops" in pk:
        out.append("FP32 alternatives (`fr_probe_fp32_paths`): FFMA2 chains %.1f TFLOP/s; with 8 integer multiply-adds beside every 16 FMAs FFMA %.1f, "
                   "FFMA2 %.1f; `mma.sync.m16n8k8` TF32 %.1f (3xTF32: %.1f of FP32-equivalent work)."
                   % (pk["ffma2_tflops"], pk["ffma_mixed_tflops"], pk["ffma2_mixed_tflops"], pk["tf32_mma_tflops"], pk["tf32_mma_tflops"] / 3))
    out.append("")
    out.append("**%.3f GDOF-RHS/s FP64** (%.2f ms per step), **%.3f FP32** (%.2f ms), end to end through `fr_rk_step_host` %.3f."
               % (d["value"], d["ms_per_step"], d["fp32"]["value"], d["fp32"]["ms_per_step"], d["e2e"]["value"]))
    out.append("")
    hdr = "| kernel | FP64 ms%s | GB/s | TF | frac | DRAM / alg | pipe %% | FP32 ms%s | GB/s | TF | frac | DRAM / alg | pipe %% |" % (
        (" (prev)" if prev else ""), (" (prev)" if prev else ""))
    out.append(hdr)
    out.append("|" + "---|" * 13)
    k64, k32 = d["kernels_f64"], d["kernels_f32"]
    tot = {"f64": 0.0, "f32": 0.0}
    for i, k in enumerate(k64):
        cells = [k["name"]]
        for prec, ks in (("f64", k64), ("f32", k32)):
            q = ks[i]
            ms = q["ms"]
            tot[prec] += ms
            gbs = q["alg_bytes"] / ms / 1e6
            tf = q["flops"] / ms / 1e9
            frac = max(gbs / hbm, tf / peak[prec])
            pm = ""
            if prev:
                pk_ = prev["kernels_" + prec]
                pm = " (%.3f)" % pk_[i]["ms"] if i < len(pk_) and pk_[i]["name"] == q["name"] else " (-)"
            t = traffic.get((prec, q["name"]))
            cells += ["%.3f%s" % (ms, pm), "%.0f" % gbs, "%.1f" % tf, "%.2f" % frac,
                      "%.2f" % (t["dram"] / q["alg_bytes"]) if t else "-",
                      "%.0f" % (t["pipe64"] if prec == "f64" else t["pipe32"]) if t else "-"]
        out.append("| " + " | ".join(cells) + " |")
    pt = ""
    if prev:
        pt = " (%.3f)"
    out.append("| total | %.3f%s | | | | | | %.3f%s | | | | | |" % (
        tot["f64"], (pt % sum(k["ms"] for k in prev["kernels_f64"])) if prev else "",
        tot["f32"], (pt % sum(k["ms"] for k in prev["kernels_f32"])) if prev else ""))
    out.append("")
    out.append("Plans chosen by `fr_setup` (`fr_plan_describe`; warps = groups x row-warps x column-warps + producers):")
    out.append("")
    out.append("```")
    out += list(d["plan"]) + list(d["fp32"]["plan"])
    out.append("```")
    sys.stdout.write("\n".join(out) + "\n")


if __name__ == "__main__":
    main()
