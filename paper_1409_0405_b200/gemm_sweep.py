"""Operator-product micro-benchmark (BASELINE.json configs[3]):  C <- c1*A*B + c2*C  (eq. 1) through `fr_gemm_plan_*`.

A: dense M x K, entries N(0,1), seeded, for each (element type in {tet, pri, hex}, p = 1..6, operator in {M0: N_f x N_u,
grad: 3N_u x N_u, div: N_u x 3N_u}); B: row-major K x N with N = 5 * N_e, entries U(-1,1); c1 = 1, c2 in {0, 1}; FP32 and FP64.
Reports achieved GB/s (algorithmic bytes (K + M (1 + [c2 != 0])) N w over CUDA-event time) and dense TFLOP/s, checks a column
sample against numpy, and -- as context only, the paper's own method -- times cuBLAS through torch.matmul.

  python -m paper_1409_0405_b200.gemm_sweep [--max-gb 6] [--neles 1000 100000 1000000] [--csv out.csv] [--summary out.md]

`plan` column: how fr_gemm_plan_create runs the operator (fr_gemm_plan_describe) -- "resident" (image in shared memory, one launch),
"resident xN" (N row blocks of A, one launch each), "streamed" / "streamed xN" (operator blocks travel through the TMA ring).
--summary writes the per-shape table at the largest N (c2 = 0) with each shape's bound and fraction of it: the HBM peak from
MEASURED_PEAKS.json (else the profiling guide's fallback), the arithmetic peaks measured by the library's probes in the same run.
"""
import argparse
import json
import os
import sys

import numpy as np

SEED = 14090408


def npts(etype, p):
    if etype == "tet":
        return (p + 1) * (p + 2) * (p + 3) // 6, 2 * (p + 1) * (p + 2)
    if etype == "pri":
        return (p + 1) ** 2 * (p + 2) // 2, (p + 1) * (p + 2) + 3 * (p + 1) ** 2
    return (p + 1) ** 3, 6 * (p + 1) ** 2


def shapes():
    for et in ("tet", "pri", "hex"):
        for p in range(1, 7):
            nu, nf = npts(et, p)
            yield et, p, "M0", nf, nu
            yield et, p, "grad", 3 * nu, nu
            yield et, p, "div", nu, 3 * nu


def plan_form(desc):
    lines = [l for l in desc.splitlines() if l.strip()]
    form = "streamed" if "streamed" in lines[0] and "register-tile" not in lines[0] else ("register-tile" if "register-tile" in lines[0] else "resident")
    return form + (" x%d" % len(lines) if len(lines) > 1 else "")


def write_summary(path, rows, cmd, hbm, hbm_src, pk64, pk32):
    """Per shape, largest N, c2 = 0: achieved GB/s and TFLOP/s, the bound by arithmetic intensity and the fraction of it."""
    best = {}
    for r in rows:
        prec, et, p, op, M, K, N, c2 = r[:8]
        if c2 != 0.0:
            continue
        key = (et, p, op, M, K)
        if key not in best:
            best[key] = {}
        if prec not in best[key] or N > best[key][prec][6]:
            best[key][prec] = r
    peak = {"f64": pk64, "f32": pk32}
    ridge = {k: peak[k] * 1e3 / hbm for k in peak}
    out = ["# Operator-product sweep of BASELINE.json configs[3] (`%s`), one B200" % os.path.basename(path).replace(".md", ".csv"), "",
           "Command: `%s` (plain run; 54 shapes x FP64/FP32 x N_e x c2 in {0, 1}; every row is checked against a float64 product on a" % cmd,
           "column sample; `fr_gemm_plan_create` times its launch geometries and, for operators larger than shared memory, the resident-row-block",
           "and the streamed form; `cublas_ms` = `torch.matmul` on the same data, context only, P:64). %d rows, all parity checks passed." % len(rows), "",
           "Largest N per shape, c2 = 0; bound by arithmetic intensity (ridge %.2f / %.2f flop/B with HBM %.0f GB/s [%s], FP64 tensor pipe %.1f and"
           % (ridge["f64"], ridge["f32"], hbm, hbm_src, pk64),
           "FP32 FFMA %.1f TFLOP/s, both measured by the library's probes in this run):" % pk32, "",
           "| type p op | M x K | FP64 plan | GB/s | TF | bound | frac | vs library | FP32 plan | GB/s | TF | bound | frac | vs library |",
           "|---|---|---|---|---|---|---|---|---|---|---|---|---|---|"]
    stats = {"f64": [], "f32": []}
    for (et, p, op, M, K), d in best.items():
        cells = ["%s %d %s" % (et, p, op), "%d x %d" % (M, K)]
        for prec in ("f64", "f32"):
            r = d[prec]
            w = 8 if prec == "f64" else 4
            gbs, tfs, ms, cms, plan = r[9], r[10], r[8], r[12], r[13]
            ai = 2.0 * M * K / ((M + K) * w)
            flop_bound = ai > ridge[prec]
            frac = tfs / peak[prec] if flop_bound else gbs / hbm
            stats[prec].append((flop_bound, frac, cms / ms))
            cells += [plan, "%.0f" % gbs, "%.1f" % tfs, "flop" if flop_bound else "hbm", "%.2f" % frac, "%.2f" % (cms / ms)]
        out.append("| " + " | ".join(cells) + " |")
    out.append("")
    for prec in ("f64", "f32"):
        st = stats[prec]
        hb = sorted(f for b, f, _ in st if not b)
        fb = sorted(f for b, f, _ in st if b)
        slow = [x for _, _, x in st if x < 1.0]
        out.append("%s: %d of %d shapes at >= 0.70 of their bound (HBM-bound shapes: median %.2f, min %.2f; compute-bound: median %.2f, min %.2f); "
                   "%d shapes slower than the library GEMM%s." % (prec.upper(), sum(f >= 0.70 for _, f, _ in st), len(st), hb[len(hb) // 2], hb[0],
                                                                  fb[len(fb) // 2], fb[0], len(slow), (" (worst %.2f x)" % min(slow)) if slow else ""))
        out.append("")
    with open(path, "w") as f:
        f.write("\n".join(out))


def main():
    import torch
    from . import binding
    ap = argparse.ArgumentParser()
    ap.add_argument("--max-gb", type=float, default=6.0, help="cap on (K + 2M) N w per case")
    ap.add_argument("--neles", type=int, nargs="+", default=[1000, 100000, 1000000])
    ap.add_argument("--csv", default=None)
    ap.add_argument("--reps", type=int, default=3)
    ap.add_argument("--summary", default=None, help="write the per-shape markdown table (largest N, c2 = 0)")
    args = ap.parse_args()
    if not torch.cuda.is_available():
        raise SystemExit("gemm_sweep needs a CUDA device (no CPU fallback)")
    rng = np.random.Generator(np.random.PCG64(SEED))
    stream = torch.cuda.current_stream().cuda_stream
    rows = []
    hdr = "prec etype p op M K N c2 ms GBs TFs err cublas_ms plan"
    print(hdr)
    for et, p, op, M, K in shapes():
        A = rng.standard_normal((M, K))
        for prec in ("f64", "f32"):
            w = 8 if prec == "f64" else 4
            tdt = torch.float64 if prec == "f64" else torch.float32
            plan = binding.GemmPlan(A, prec)
            form = plan_form(plan.describe())
            dA = torch.from_numpy(A).to(tdt).cuda()
            for ne in args.neles:
                N = 5 * ne
                cap = int(args.max_gb * 1e9 / ((K + 2 * M) * w))
                N = max(20, min(N, cap) // 20 * 20)   # multiple of 5 (variables) and of 4 (16-byte rows)
                B = torch.rand((K, N), dtype=tdt, device="cuda") * 2 - 1
                for c2 in (0.0, 1.0):
                    C0 = torch.rand((M, N), dtype=tdt, device="cuda") * 2 - 1
                    C = C0.clone()
                    plan.run(B.data_ptr(), N, C.data_ptr(), N, N, c1=1.0, c2=c2, stream=stream)
                    torch.cuda.synchronize()
                    ns = min(N, 512)
                    ref = dA.double()[:, :] @ B[:, :ns].double() + c2 * C0[:, :ns].double()
                    scale = (dA.double().abs() @ B[:, :ns].double().abs() + abs(c2) * C0[:, :ns].double().abs()).max().item()
                    err = (C[:, :ns].double() - ref).abs().max().item() / scale
                    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
                    e0.record()
                    for _ in range(args.reps):
                        plan.run(B.data_ptr(), N, C.data_ptr(), N, N, c1=1.0, c2=c2, stream=stream)
                    e1.record()
                    e1.synchronize()
                    ms = e0.elapsed_time(e1) / args.reps
                    # context: cuBLAS via torch (c2 = 0 form only)
                    cms = float("nan")
                    if c2 == 0.0:
                        torch.matmul(dA, B, out=C)
                        e0.record()
                        for _ in range(args.reps):
                            torch.matmul(dA, B, out=C)
                        e1.record()
                        e1.synchronize()
                        cms = e0.elapsed_time(e1) / args.reps
                    nbytes = (K + M * (2 if c2 else 1)) * N * w
                    r = (prec, et, p, op, M, K, N, c2, ms, nbytes / ms / 1e6, 2.0 * M * K * N / ms / 1e9, err, cms, form)
                    rows.append(r)
                    print("%s %s %d %s %d %d %d %.0f %.4f %.0f %.2f %.1e %.4f %s" % r, flush=True)
                    tol = 1e-13 if prec == "f64" else 1e-5
                    assert err <= tol, "parity failure: %r" % (r,)
                    del C, C0
                del B
            plan.close()
    if args.summary:
        root = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
        try:
            with open(os.path.join(root, "MEASURED_PEAKS.json")) as f:
                hbm, hbm_src = float(json.load(f)["hbm_gbs"]), "MEASURED_PEAKS.json"
        except Exception:
            hbm, hbm_src = 6550.0, "B200_PROFILING.md fallback"
        pk = binding.probe_peaks()
        write_summary(args.summary, rows, "python -m paper_1409_0405_b200.gemm_sweep " + " ".join(sys.argv[1:]), hbm, hbm_src,
                      binding.probe_dmma(), pk["fp32_tflops"])
    if args.csv:
        with open(args.csv, "w") as f:
            f.write(hdr.replace(" ", ",") + "\n")
            for r in rows:
                f.write(",".join(str(x) for x in r) + "\n")


if __name__ == "__main__":
    sys.exit(main())
