"""CPU checks of the measurement tools that write what `profiles/` keeps: the per-kernel roofline table (`kernel_table`), the ncu
launch-list table (`ncu_summary --launches`) and the operator-product sweep's summary (`gemm_sweep.write_summary`).  They only
rearrange numbers a GPU run produced; here they run on small hand-made inputs and the arithmetic of their columns is checked."""
import json
import os
import subprocess
import sys

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _bench_line():
    def k(name, ms, gb, gf):
        return dict(name=name, ms=ms, alg_bytes=gb * 1e9, flops=gf * 1e9, category=0)
    k64 = [k("tet:S1_M0", 0.5, 2.0, 10.0), k("S7_comm_flux", 1.0, 5.0, 1.0)]
    k32 = [k("tet:S1_M0", 0.25, 1.0, 10.0), k("S7_comm_flux", 0.5, 2.5, 1.0)]
    return dict(metric="GDOF-RHS/s", value=2.0, ms_per_step=50.0, e2e=dict(value=1.0),
                roofline=dict(hbm=dict(peak=5000.0, peak_source="test")),
                peaks=dict(fp64_tensor_tflops=40.0, fp32_ffma_tflops=80.0),
                kernels_f64=k64, kernels_f32=k32, plan=["f64 plan line"],
                fp32=dict(value=3.0, ms_per_step=30.0, plan=["f32 plan line"]))


def test_kernel_table_fractions_and_traffic(tmp_path):
    b = tmp_path / "bench.json"
    b.write_text("noise\n" + json.dumps(_bench_line()) + "\n")
    t = tmp_path / "traffic.csv"
    t.write_text("f64,tet:S1_M0,3000000000,0.5,100,200.0,80.0,1.0,k\nf64,S7_comm_flux,6500000000,1.0,120,0,0,0,k\n"
                 "f32,tet:S1_M0,1000000000,0.25,100,200.0,0,50.0,k\nf32,S7_comm_flux,2500000000,0.5,80,0,0,10.0,k\n")
    out = subprocess.run([sys.executable, "-m", "paper_1409_0405_b200.kernel_table", str(b), "--traffic", str(t), "--prev", str(b)],
                         cwd=ROOT, capture_output=True, text=True, check=True).stdout
    rows = {l.split("|")[1].strip(): [c.strip() for c in l.split("|")[2:-1]] for l in out.splitlines() if l.startswith("| ")}
    s1 = rows["tet:S1_M0"]
    # FP64: 2 GB / 0.5 ms = 4000 GB/s = 0.80 of 5000; 10 GF / 0.5 ms = 20 TF = 0.50 of 40 -> frac 0.80; DRAM / alg = 1.50; pipe 80
    assert s1[0] == "0.500 (0.500)" and s1[1] == "4000" and s1[2] == "20.0" and s1[3] == "0.80" and s1[4] == "1.50" and s1[5] == "80"
    # FP32: 1 GB / 0.25 ms = 4000 GB/s (0.80); 40 TF of 80 (0.50)
    assert s1[7] == "4000" and s1[8] == "40.0" and s1[9] == "0.80" and s1[10] == "1.00" and s1[11] == "50"
    s7 = rows["S7_comm_flux"]
    assert s7[1] == "5000" and s7[3] == "1.00" and s7[4] == "1.30"
    assert rows["total"][0] == "1.500 (1.500)" and rows["total"][6] == "0.750 (0.750)"
    assert "f64 plan line" in out and "f32 plan line" in out


def test_launch_table(tmp_path):
    from paper_1409_0405_b200 import ncu_summary
    hdr = '"ID","Process ID","Process Name","Host Name","Kernel Name","Context","Stream","Block Size","Grid Size","Device","CC","Section Name","Metric Name","Metric Unit","Metric Value"'
    def row(i, name, block, ns):
        return '"%d","1","python","h","void unnamed>::%s(unnamed>::Args<T1>)","1","13","(%d, 1, 1)","(148, 1, 1)","0","10.0","s","gpu__time_duration.sum","ns","%d"' % (i, name, block, ns)
    p = tmp_path / "l.csv"
    p.write_text("==PROF== noise\n" + "\n".join([hdr, row(0, "k_a<double>", 128, 1000000), row(1, "k_b<double, 3, 1>", 352, 3000000),
                                                 row(2, "k_a<double>", 128, 2000000)]) + "\n")
    md = ncu_summary.launch_table(str(p)).splitlines()
    assert md[2].startswith("| `k_a<double>` x128 | 2 | 3.000 | 50.0 % | 1.500 |") or md[3].startswith("| `k_a<double>` x128 | 2 | 3.000 | 50.0 % | 1.500 |")
    assert any(l.startswith("| `k_b<double, 3, 1>` x352 | 1 | 3.000 | 50.0 % | 3.000 |") for l in md)
    assert md[-1] == "| total | 3 | 6.000 | | |"


def test_gemm_sweep_summary_and_plan_form(tmp_path):
    from paper_1409_0405_b200 import gemm_sweep as G
    assert G.plan_form("f64 rows 0..215 of 216x648 dense, streamed warps=1x7x1+1\n") == "streamed"
    assert G.plan_form("a dense\nb dense\nc dense\n") == "resident x3"
    assert G.plan_form("f64 343x343 register-tile kernel TY=8 MT=16\n") == "register-tile"
    rows = []
    for et, p, op, M, K in G.shapes():
        for prec, w in (("f64", 8), ("f32", 4)):
            for N in (5000, 500000):
                ms = 1.0
                rows.append((prec, et, p, op, M, K, N, 0.0, ms, (M + K) * N * w / ms / 1e6, 2.0 * M * K * N / ms / 1e9, 1e-16, 2.0, "resident"))
                rows.append((prec, et, p, op, M, K, N, 1.0, ms, 0.0, 0.0, 1e-16, float("nan"), "resident"))
    out = tmp_path / "s.md"
    G.write_summary(str(out), rows, "cmd", 6000.0, "test", 40.0, 80.0)
    txt = out.read_text()
    lines = [l for l in txt.splitlines() if l.startswith("| ")]
    assert len(lines) == 1 + 54                           # header + 54 shapes (3 types x p = 1..6 x 3 operators)
    cells = [c.strip() for c in [l for l in lines if l.startswith("| tet 1 M0 ")][0].split("|")[1:-1]]
    # tet p = 1 M0: 12 x 4, N = 500000 (the largest): GB/s = 16 * 5e5 * 8 / 1 ms = 64 -> hbm-bound (AI 0.75 < ridge 6.7), frac 64/6000
    assert cells[1] == "12 x 4" and cells[3] == "64" and cells[5] == "hbm" and cells[6] == "0.01" and cells[7] == "2.00"
    # hex p = 6 grad, 1029 x 343: 2 * 1029 * 343 * 5e5 / 1 ms = 353 TFLOP/s, "8.82" of the 40 TFLOP/s test peak: compute-bound
    big = [c.strip() for c in [l for l in lines if l.startswith("| hex 6 grad ")][0].split("|")[1:-1]]
    assert big[5] == "flop" and big[6] == "8.82"
    assert "of 54 shapes at >= 0.70 of their bound" in txt and "0 shapes slower than the library GEMM" in txt
