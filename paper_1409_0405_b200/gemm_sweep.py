"""Operator-product micro-benchmark (BASELINE.json configs[3]):  C <- c1*A*B + c2*C  (eq. 1) through `fr_gemm_plan_*`.

A: dense M x K, entries N(0,1), seeded, for each (element type in {tet, pri, hex}, p = 1..6, operator in {M0: N_f x N_u,
grad: 3N_u x N_u, div: N_u x 3N_u}); B: row-major K x N with N = 5 * N_e, entries U(-1,1); c1 = 1, c2 in {0, 1}; FP32 and FP64.
Reports achieved GB/s (algorithmic bytes (K + M (1 + [c2 != 0])) N w over CUDA-event time) and dense TFLOP/s, checks a column
sample against numpy, and -- as context only, the paper's own method -- times cuBLAS through torch.matmul.

  python -m paper_1409_0405_b200.gemm_sweep [--max-gb 6] [--neles 1000 100000 1000000] [--csv out.csv]
"""
import argparse
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


def main():
    import torch
    from . import binding
    ap = argparse.ArgumentParser()
    ap.add_argument("--max-gb", type=float, default=6.0, help="cap on (K + 2M) N w per case")
    ap.add_argument("--neles", type=int, nargs="+", default=[1000, 100000, 1000000])
    ap.add_argument("--csv", default=None)
    ap.add_argument("--reps", type=int, default=3)
    args = ap.parse_args()
    if not torch.cuda.is_available():
        raise SystemExit("gemm_sweep needs a CUDA device (no CPU fallback)")
    rng = np.random.Generator(np.random.PCG64(SEED))
    stream = torch.cuda.current_stream().cuda_stream
    rows = []
    hdr = "prec etype p op M K N c2 ms GBs TFs err cublas_ms"
    print(hdr)
    for et, p, op, M, K in shapes():
        A = rng.standard_normal((M, K))
        for prec in ("f64", "f32"):
            w = 8 if prec == "f64" else 4
            tdt = torch.float64 if prec == "f64" else torch.float32
            plan = binding.GemmPlan(A, prec)
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
                    r = (prec, et, p, op, M, K, N, c2, ms, nbytes / ms / 1e6, 2.0 * M * K * N / ms / 1e9, err, cms)
                    rows.append(r)
                    print("%s %s %d %s %d %d %d %.0f %.4f %.0f %.2f %.1e %.4f" % r, flush=True)
                    tol = 1e-13 if prec == "f64" else 1e-5
                    assert err <= tol, "parity failure: %r" % (r,)
                    del C, C0
                del B
            plan.close()
    if args.csv:
        with open(args.csv, "w") as f:
            f.write(hdr.replace(" ", ",") + "\n")
            for r in rows:
                f.write(",".join(str(x) for x in r) + "\n")


if __name__ == "__main__":
    sys.exit(main())
