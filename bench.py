#!/usr/bin/env python
"""bench.py -- throughput of the flux-reconstruction hot path on B200 (contract: see DESIGN.md "Measurement").

Workload (BASELINE.json configs[2], "RK45 stages timed"): the synthetic cylinder-like O-mesh of 120 000 prisms +
360 000 tetrahedra at p = 4 (21.6 M solution points), compressible Navier-Stokes at Re = 3900, M = 0.2, Rusanov +
LDG, RK45[2R+].  One "step" = one RK45[2R+] time step = 5 evaluations of the whole right-hand side (S1..S10 of
SURVEY 8(a)) through the C ABI (`fr_rk_step`).  metric = GDOF-RHS/s = solution points x RHS evaluations / s / 1e9.

  python bench.py [--gpus N] [--steps K] [--warmup W] [--impl frb200|reference] [--small]
                  [--workload config3|config2|config5] [--kernels] [--no-gemm] [--no-cpu-baseline]

`--workload config5` is BASELINE.json configs[4] (the config-3 generator scaled to ~150 GB of HBM, p = 3, FP32 only: takes
about four minutes of host-side mesh generation and set-up before the timed steps); `--workload config2` the 32^3 mixed
periodic box at p = 4.  The default line also carries a `gemm` object: the operator product of PAPER.md:37 eq. 1 alone
(`fr_gemm_plan_*`) on representative shapes of BASELINE.json configs[3], with the same-box library GEMM as context.

`--impl reference` times the CPU oracle (oracle/fr_oracle.py, FP64 numpy, as it stands) on the host cores on a
bounded sample of the same workload.  Under torchrun each rank runs an independent replica (DESIGN.md "Multi-GPU":
replicas only, no collective on the data path).
"""
import argparse
import json
import os
import subprocess
import sys
import threading
import time

ROOT = os.path.dirname(os.path.abspath(__file__))
sys.path.insert(0, ROOT)

import numpy as np  # noqa: E402

METRIC = "GDOF-RHS/s"
FULL = dict(p=4, ntheta=100, nz=15, nlayers=40, nr=40)      # BASELINE.json configs[2]
SMALL = dict(p=4, ntheta=24, nz=4, nlayers=10, nr=10)       # --small: quick functional check only
SAMPLE = dict(p=4, ntheta=40, nz=6, nlayers=40, nr=40)      # bounded sample for the CPU oracle (16 % of FULL)
DT = 2e-6


def _peaks():
    """Roofline denominators: MEASURED_PEAKS.json (driver-written) else the profiling guide's fallback."""
    path = os.path.join(ROOT, "MEASURED_PEAKS.json")
    try:
        with open(path) as f:
            d = json.load(f)
        return float(d["hbm_gbs"]), "MEASURED_PEAKS.json hbm_gbs"
    except Exception:
        return 6550.0, "fallback (B200_PROFILING.md measured copy rate)"


class ClockSampler(threading.Thread):
    """Samples SM clock and throttle reasons with nvidia-smi while the timed region runs."""

    def __init__(self, index=0, period=0.2):
        super().__init__(daemon=True)
        self.index, self.period = index, period
        self.samples, self.reasons, self.maxmhz = [], set(), None
        self._stop_evt = threading.Event()

    def _query(self):
        q = "clocks.sm,clocks.max.sm,clocks_event_reasons.active"
        try:
            out = subprocess.run(["nvidia-smi", "-i", str(self.index), "--query-gpu=" + q, "--format=csv,noheader,nounits"],
                                 capture_output=True, text=True, timeout=5).stdout.strip()
            a = [x.strip() for x in out.split(",")]
            self.samples.append(float(a[0]))
            self.maxmhz = float(a[1])
            bits = int(a[2], 16)
            names = {0x1: "gpu_idle", 0x2: "applications_clocks_setting", 0x4: "sw_power_cap", 0x8: "hw_slowdown",
                     0x10: "sync_boost", 0x20: "sw_thermal_slowdown", 0x40: "hw_thermal_slowdown",
                     0x80: "hw_power_brake_slowdown", 0x100: "display_clock_setting"}
            for b, n in names.items():
                if bits & b and n != "gpu_idle":
                    self.reasons.add(n)
        except Exception:
            pass

    def run(self):
        while not self._stop_evt.is_set():
            self._query()
            self._stop_evt.wait(self.period)

    def stop(self):
        self._stop_evt.set()
        self.join(timeout=10)
        s = sorted(self.samples)
        return dict(sm_mhz=(s[len(s) // 2] if s else None), sm_max_mhz=self.maxmhz, reasons=sorted(self.reasons),
                    samples=len(s))


CONFIG5 = dict(scale=2, copies=9, p=3)                       # BASELINE.json configs[4]: 4.32 M prisms + 12.96 M tetrahedra, ~156 GB
CONFIG2 = dict(n=32, p=4)                                    # BASELINE.json configs[1] at its largest sweep size


def _case(kind):
    from fr_inputs import cases
    if "copies" in kind:
        c = cases.config3(p=kind["p"], ntheta=100 * kind["scale"], nz=15 * kind["scale"], seed=cases.SEEDS["c5"])
        return cases.replicate(c, kind["copies"], amp=0.005, seed=cases.SEEDS["c5"], compact=True)
    if "n" in kind:
        return cases.config2(kind["n"], kind["p"], "ns", numbering="morton")      # Morton order is the primary numbering for throughput
    return cases.config3(**kind)


def _workload_name(kind, case):
    ne = {e["etype"]: e["neles"] for e in case["eles"]}
    if "copies" in kind:
        return "config5: config-3 generator x%d held as %d disjoint copies, p=%d NS RK45[2R+]: %d pri + %d tet" % (
            kind["scale"], kind["copies"], kind["p"], ne.get("pri", 0), ne.get("tet", 0))
    if "n" in kind:
        return "config2 periodic mixed box %d^3 p=%d NS RK45[2R+] vortex: %d pri + %d tet" % (kind["n"], kind["p"], ne.get("pri", 0), ne.get("tet", 0))
    return "config3 cylinder O-mesh p=%d NS RK45[2R+]: %d pri + %d tet" % (kind["p"], ne.get("pri", 0), ne.get("tet", 0))


# ------------------------------------------------------------------------------------------------ CPU oracle arm
def oracle_rate(case, nrhs, budget_s=40.0):
    """GDOF-RHS/s of the oracle as it stands on this host: `nrhs` RHS evaluations (at least one)."""
    from fr_inputs import cases
    from oracle import fr_oracle as O
    n = cases.ndof(case)
    t0 = time.perf_counter()
    done = 0
    us = case["u0"]
    for _ in range(max(1, nrhs)):
        O.rhs(case["cfg"], case["eles"], case["ifc"], case["bcs"], us)
        done += 1
        if time.perf_counter() - t0 > budget_s:
            break
    dt = time.perf_counter() - t0
    return n * done / dt / 1e9, done, dt


def _blas_threads():
    try:
        from threadpoolctl import threadpool_info
        return max([i.get("num_threads", 1) for i in threadpool_info()] + [1])
    except Exception:
        return os.cpu_count() or 1


def _cpu_model():
    try:
        with open("/proc/cpuinfo") as f:
            for line in f:
                if line.startswith("model name"):
                    return line.split(":", 1)[1].strip()
    except Exception:
        pass
    return "unknown"


def oracle_rate_single_thread(case):
    """The same oracle with the BLAS pool limited to one thread (so the figure can be scaled)."""
    try:
        from threadpoolctl import threadpool_limits
        with threadpool_limits(limits=1):
            return oracle_rate(case, 1, budget_s=30.0)
    except Exception:
        return None


def run_reference(args):
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    kind = SMALL if args.small else SAMPLE
    case = _case(kind)
    from fr_inputs import cases
    for _ in range(args.warmup and 1):
        oracle_rate(case, 1)
    # one "step" of this arm = one RHS evaluation of the bounded sample (an RK45 step is 5 of them)
    rate, done, dt = oracle_rate(case, args.steps, budget_s=150.0)
    cores = _blas_threads()
    sample = "%s (%d DOF, %.0f %% of the full workload), %d RHS evaluations" % (
        _workload_name(kind, case), cases.ndof(case), 100.0 * cases.ndof(case) / 21.6e6, done)
    line = dict(impl="reference", metric=METRIC, value=rate, unit="GDOF-RHS/s", n_gpus=args.gpus, steps=done,
                warmup=args.warmup, ms_per_step=1e3 * dt / done, higher_is_better=True, scaling="weak", vs_baseline=None,
                dtype="f64", data="synthetic",
                config=dict(workload=_workload_name(FULL if not args.small else SMALL, case), sample=sample),
                cpu_baseline=dict(value=rate, unit="GDOF-RHS/s", cores=cores, kind="oracle", sample=sample),
                e2e=dict(value=rate, unit="GDOF-RHS/s", h2d_bytes_per_step=0, d2h_bytes_per_step=0), gpu_launches=0)
    print(json.dumps(line))


# ------------------------------------------------------------------------------------------------ CUDA arm
def max_over_ranks(seconds, world, dist, torch, device):
    """Replicas only: every rank times the same work on its own GPU; the job's time is the slowest rank's."""
    if world <= 1:
        return seconds
    t = torch.tensor([seconds], dtype=torch.float64, device=device)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())


def aggregate_rate(ndof, rhs_per_step, steps, seconds, world):
    """Whole-job GDOF-RHS/s: the units all `world` replicas processed over the max-over-ranks time."""
    return world * ndof * rhs_per_step * steps / seconds / 1e9


def _time_steps(ctx, stream, dt, steps, torch):
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    e0.record(stream)
    ctx.rk_run(dt, steps)
    e1.record(stream)
    e1.synchronize()
    return e0.elapsed_time(e1) * 1e-3


def _measure(case, prec, args, torch, dist, rank, world, with_e2e=True, sampler=None, profiler=False):
    from fr_inputs import cases
    from paper_1409_0405_b200 import Context
    stream = torch.cuda.Stream()
    ctx = Context(case, prec=prec, stepper="rk45", stream=stream.cuda_stream)
    ndof = cases.ndof(case)
    ctx.set_state(case["u0"])
    ctx.rk_run(DT, args.warmup)
    ctx.sync()
    n0 = ctx.launch_count()
    if world > 1:
        dist.barrier()
    torch.cuda.synchronize()
    if sampler is not None:
        sampler.start()
    # `ncu --profile-from-start off` captures exactly the timed region of one context (--profile-prec; set-up launches candidate
    # geometries for autotuning, which must not end up in the launch list)
    if profiler:
        torch.cuda.cudart().cudaProfilerStart()
    sec = _time_steps(ctx, stream, DT, args.steps, torch)
    torch.cuda.synchronize()
    if profiler:
        torch.cuda.cudart().cudaProfilerStop()
    clocks = sampler.stop() if sampler is not None else None
    launches = ctx.launch_count() - n0
    sec = max_over_ranks(sec, world, dist, torch, "cuda")
    nstage = 5
    res = dict(seconds=sec, value=aggregate_rate(ndof, nstage, args.steps, sec, world), launches=launches, clocks=clocks,
               ndof=ndof)
    # state must still be finite after the timed steps (a blown-up run would be timing NaN arithmetic)
    chk = ctx.get_state()
    res["finite"] = bool(all(np.isfinite(a).all() for a in chk))
    # per-kernel CUDA-event breakdown of one RHS as an RK stage runs it (same context, same data, right after the timed region)
    res["kernels"] = ctx.profile_stage_kernels(reps=3)
    res["plan"] = ctx.plan_describe()
    if with_e2e:
        # end to end through the C ABI with HOST buffers: H2D of the state, one RK45 step, D2H of the new state
        tdt = torch.float64 if prec == "f64" else torch.float32
        hbuf = []
        for u, ld in zip(chk, ctx.ld):
            h = torch.zeros((u.shape[0], 5, ld), dtype=tdt).pin_memory()
            h[:, :, :u.shape[2]] = torch.from_numpy(np.ascontiguousarray(u)).to(tdt)
            hbuf.append(h)
        ptrs = [h.data_ptr() for h in hbuf]
        ne2e = max(2, min(args.steps, 5))
        ctx.rk_step_host(DT, ptrs)
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()
        t0 = time.perf_counter()
        for _ in range(ne2e):
            ctx.rk_step_host(DT, ptrs)
        torch.cuda.synchronize()
        t1 = time.perf_counter() - t0
        t1 = max_over_ranks(t1, world, dist, torch, "cuda")
        nb = int(sum(h.numel() * h.element_size() for h in hbuf))
        res["e2e"] = dict(value=aggregate_rate(ndof, nstage, ne2e, t1, world), unit="GDOF-RHS/s", h2d_bytes_per_step=nb,
                          d2h_bytes_per_step=nb, steps=ne2e)
    ctx.close()
    return res


def _traffic(name, prec):
    """DRAM bytes per launch of kernel `name` from the committed ncu --set full summary (profiles/r02_traffic.csv, written by
    `python -m paper_1409_0405_b200.ncu_summary`; the capture command is in profiles/r02_traffic.md), else None."""
    try:
        with open(os.path.join(ROOT, "profiles", "r02_traffic.csv")) as f:
            for line in f:
                a = line.strip().split(",")
                if len(a) >= 3 and a[0] == prec and a[1] == name:
                    return float(a[2])
    except Exception:
        pass
    return None


# arithmetic peaks: measured live by the library's own probes (fr_probe_dmma: FP64 tensor pipe, mma.m8n8k4.f64 chains;
# fr_probe_peaks: FP32 FFMA chains) at the start of the run and recorded in the line.  The HBM peak comes from MEASURED_PEAKS.json.
FLOP_PEAK = {}


def _probe_flop_peaks():
    from paper_1409_0405_b200 import binding
    pk = binding.probe_peaks()
    dm = binding.probe_dmma()
    FLOP_PEAK["f64"] = (dm, "tensor", "fr_probe_dmma (mma.m8n8k4.f64 chains), measured in this run")
    FLOP_PEAK["f32"] = (pk["fp32_tflops"], "alu", "fr_probe_peaks (FFMA chains), measured in this run")
    alt = binding.probe_fp32_paths()   # FFMA2 (what the FP32 products issue), the same beside integer work, legacy TF32 mma
    return dict(fp64_tensor_tflops=dm, fp64_dfma_tflops=pk["fp64_tflops"], fp32_ffma_tflops=pk["fp32_tflops"], copy_gbs=pk["copy_gbs"], **alt)


def _groups(kernels):
    """Per-kernel-group milliseconds of one right-hand side (BASELINE.json configs[4]: "GEMM vs flux vs interface")."""
    names = {0: "operator_products_incl_fused_pointwise_ms", 1: "pointwise_flux_ms", 2: "interface_ms"}
    g = {v: 0.0 for v in names.values()}
    for k in kernels:
        g[names[k["category"]]] += k["ms"]
    g["total_ms"] = sum(g.values())
    return g


def _roofline(kernels, peak, peak_src, prec="f64"):
    """Dominant kernel of one RHS by CUDA-event time.  Its bound is decided by its arithmetic intensity (dense flops over
    algorithmic bytes) against the ridge of the measured peaks; achieved = algorithmic bytes (or flops) per launch / mean duration."""
    tot = sum(k["ms"] for k in kernels)
    top = max(kernels, key=lambda k: k["ms"])
    sec = top["ms"] * 1e-3
    gbs = top["alg_bytes"] / sec / 1e9
    tfl = top["flops"] / sec / 1e12
    fpeak, fbound, fsrc = FLOP_PEAK[prec]
    ridge = fpeak * 1e12 / (peak * 1e9)
    ai = top["flops"] / max(top["alg_bytes"], 1.0)
    whole = sum(k["alg_bytes"] for k in kernels) / (tot * 1e-3) / 1e9
    common = dict(kernel=top["name"], traffic=_traffic(top["name"], prec), share_of_rhs=top["ms"] / tot, ms_per_launch=top["ms"],
                  alg_bytes_per_launch=top["alg_bytes"], flops_per_launch=top["flops"], intensity_flop_per_byte=ai, ridge=ridge,
                  hbm=dict(achieved=gbs, peak=peak, unit="GB/s", frac=gbs / peak, peak_source=peak_src),
                  flop=dict(achieved=tfl, peak=fpeak, unit="TFLOP/s", frac=tfl / fpeak, peak_source=fsrc),
                  whole_rhs=dict(alg_gbs=whole, frac=whole / peak, ms=tot,
                                 tflops=sum(k["flops"] for k in kernels) / (tot * 1e-3) / 1e12))
    if ai > ridge:
        return dict(bound=fbound, achieved=tfl, peak=fpeak, unit="TFLOP/s", frac=tfl / fpeak, peak_source=fsrc, **common)
    return dict(bound="hbm", achieved=gbs, peak=peak, unit="GB/s", frac=gbs / peak, peak_source=peak_src, **common)


# representative shapes of BASELINE.json configs[3]: (label, M, K); dense N(0,1) operators, B ~ U(-1,1), c1 = 1, c2 = 0
GEMM_SHAPES = [("tet p3 M0", 40, 20), ("tet p4 grad", 105, 35), ("tet p4 div", 35, 105), ("pri p3 M0", 68, 40),
               ("pri p4 div", 75, 225), ("hex p3 grad", 192, 64), ("hex p4 M0", 150, 125), ("hex p5 grad", 648, 216)]


def _gemm_sweep(torch, peak, nele=1000000, reps=10):
    """Operator product alone through fr_gemm_plan_* (C ABI), CUDA events on the launching stream; same-box torch.matmul (the
    library GEMM the paper's CUDA backend would call) as context.  N = 5 * nele columns, capped so that B and C
    stay below 24 GB."""
    from fr_inputs import cases
    from paper_1409_0405_b200 import binding
    out = []
    rng = np.random.Generator(np.random.PCG64(cases.SEEDS["c4"]))
    stream = torch.cuda.current_stream()
    for label, M, K in GEMM_SHAPES:
        A = rng.standard_normal((M, K))
        for prec, tdt, w in (("f64", torch.float64, 8), ("f32", torch.float32, 4)):
            ne = int(min(nele, 24e9 / ((M + K) * 5 * w)) // 128 * 128)
            N = 5 * ne
            B = torch.rand((K, N), dtype=tdt, device="cuda") * 2 - 1
            Cm = torch.empty((M, N), dtype=tdt, device="cuda")
            plan = binding.GemmPlan(A, prec)
            e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)

            def timed(f):
                for _ in range(3):
                    f()
                e0.record(stream)
                for _ in range(reps):
                    f()
                e1.record(stream)
                e1.synchronize()
                return e0.elapsed_time(e1) / reps
            ms = timed(lambda: plan.run(B.data_ptr(), N, Cm.data_ptr(), N, N, stream=stream.cuda_stream))
            Ad = torch.from_numpy(A).to(tdt).cuda()
            torch.backends.cuda.matmul.allow_tf32 = False
            ms_lib = timed(lambda: torch.matmul(Ad, B, out=Cm))
            plan.close()
            nbytes = (M + K) * N * w
            flops = 2.0 * M * K * N
            fpeak = FLOP_PEAK[prec][0]
            gbs, tfl = nbytes / ms / 1e6, flops / ms / 1e9
            bound = "hbm" if flops / nbytes < fpeak * 1e12 / (peak * 1e9) else FLOP_PEAK[prec][1]
            out.append(dict(shape=label, M=M, K=K, N=N, dtype=prec, ms=ms, gbs=gbs, tflops=tfl, bound=bound,
                            frac=(gbs / peak if bound == "hbm" else tfl / fpeak), library_gemm_ms=ms_lib))
            del B, Cm, Ad
    return out


def run_frb200(args):
    import torch
    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device (there is no CPU fallback; use --impl reference for the oracle)")
    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    torch.cuda.set_device(local)
    dist = None
    if world > 1:
        import torch.distributed as dist
        dist.init_process_group("nccl", device_id=torch.device("cuda", local))
    kind = SMALL if args.small else {"config3": FULL, "config5": CONFIG5, "config2": CONFIG2}[args.workload]
    case = _case(kind)
    peak, peak_src = _peaks()
    probes = _probe_flop_peaks()
    sampler = ClockSampler(index=local) if rank == 0 else None
    only32 = "copies" in kind                      # config 5 is an FP32 workload (BASELINE.json configs[4]) and fills HBM once
    if only32:
        r32 = _measure(case, "f32", args, torch, dist, rank, world, sampler=sampler, profiler=args.profile_prec == "f32")
        r64 = None
    else:
        r64 = _measure(case, "f64", args, torch, dist, rank, world, sampler=sampler, profiler=args.profile_prec == "f64")
        r32 = _measure(case, "f32", args, torch, dist, rank, world, with_e2e=False, profiler=args.profile_prec == "f32")
    if rank == 0:
        cpu = None
        if world == 1 and not args.no_cpu_baseline:
            scase = case if args.small else _case(SAMPLE)
            from fr_inputs import cases
            v, done, dt = oracle_rate(scase, 2, budget_s=20.0)
            one = oracle_rate_single_thread(_case(SMALL))
            cpu = dict(value=v, unit="GDOF-RHS/s", cores=_blas_threads(), kind="oracle", cpu_model=_cpu_model(),
                       sample="%s (%d DOF), %d RHS evaluations in %.1f s" % (
                           _workload_name(SMALL if args.small else SAMPLE, scase), cases.ndof(scase), done, dt),
                       single_thread=(dict(value=one[0], unit="GDOF-RHS/s", sample="--small mesh, 1 RHS evaluation in %.1f s, BLAS pool limited to 1 thread" % one[2])
                                      if one else None))
        main = r32 if only32 else r64
        ms = 1e3 * main["seconds"] / args.steps
        state_gb = sum(e["nupts"] * 5 * e["neles"] for e in case["eles"]) * (4 if only32 else 8) / 1e9
        line = dict(metric=METRIC, value=main["value"], unit="GDOF-RHS/s", n_gpus=world, steps=args.steps,
                    warmup=args.warmup, ms_per_step=ms, higher_is_better=True, scaling="weak", vs_baseline=None,
                    dtype="f32" if only32 else "f64", data="synthetic",
                    config=dict(workload=_workload_name(kind, case), dof=main["ndof"], rhs_per_step=5, dt=DT,
                                parallelism="replicas only: %d independent copies of the workload, no data-path collective" % world
                                if world > 1 else "single GPU",
                                l2="state %.2f GB per register, working set >> 126 MB L2: no flush needed" % state_gb),
                    clocks=main["clocks"], e2e=main.get("e2e"), gpu_launches=main["launches"],
                    roofline=_roofline(main["kernels"], peak, peak_src, "f32" if only32 else "f64"), cpu_baseline=cpu,
                    finite=main["finite"], peaks=probes, plan=main["plan"].splitlines())
        if not only32:
            line["fp32"] = dict(value=r32["value"], unit="GDOF-RHS/s", ms_per_step=1e3 * r32["seconds"] / args.steps,
                                dtype="f32", gpu_launches=r32["launches"], finite=r32["finite"],
                                roofline=_roofline(r32["kernels"], peak, peak_src, "f32"), plan=r32["plan"].splitlines())
        line["kernel_groups"] = _groups(main["kernels"])
        if world == 1 and not args.no_gemm and not args.small:
            line["gemm"] = _gemm_sweep(torch, peak)
        if args.kernels:
            if r64:
                line["kernels_f64"] = r64["kernels"]
            line["kernels_f32"] = r32["kernels"]
        print(json.dumps(line))
    if world > 1:
        dist.barrier()
        dist.destroy_process_group()


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=10)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="frb200", choices=["frb200", "reference"])
    ap.add_argument("--small", action="store_true", help="small mesh (functional check, not a bench number)")
    ap.add_argument("--kernels", action="store_true", help="add the per-kernel breakdown to the JSON line")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-gemm", action="store_true", help="skip the operator-product sweep (the `gemm` object)")
    ap.add_argument("--workload", default="config3", choices=["config3", "config2", "config5"])
    ap.add_argument("--profile-prec", default="f64", choices=["f64", "f32"],
                    help="which context's timed region cudaProfilerStart/Stop brackets (for ncu --profile-from-start off)")
    args = ap.parse_args()
    args.warmup = max(args.warmup, 3) if args.impl == "frb200" else args.warmup
    if args.impl == "reference":
        run_reference(args)
    else:
        run_frb200(args)


if __name__ == "__main__":
    main()
