"""Sustained time-marching run (BASELINE.json configs[4]): the cylinder-like O-mesh of config 3, scaled up, p = 3, FP32 (or FP64),
RK45[2R+] with fixed dt replayed as CUDA graphs (`fr_rk_run`) for `--steps` steps.  Reports GDOF-RHS/s, the totals of the five
conserved quantities and the kinetic energy (quadrature-weighted, accumulated in FP64 on the host from `fr_get_state`) at steps
0 / 10 / 100 / 1000, and the per-kernel-group time breakdown of one right-hand side (`fr_profile_rhs`: operator products incl. fused
point-wise work, stand-alone point-wise kernels, interface kernels).

  python -m paper_1409_0405_b200.sustained [--scale 2] [--copies 1] [--p 3] [--prec f32] [--steps 1000] [--dt 4e-6]
                                           [--json out.json] [--mesh cylinder|cylinder-quadratic|hex] [--n 40]

`--scale s` multiplies the circumferential and spanwise cell counts of config 3 (100 x 15) by s: elements = 480 000 s^2.  Config 5
itself is s = 6 (17.3 M elements, ~150 GB); the mesh generator is host-side numpy and its memory and time, not the library,
bound s.  `--copies K` reaches that size another way (`fr_inputs.cases.replicate`): K disjoint copies of the scale-s mesh as one
case, each with its own seeded perturbation -- s = 2, K = 9 has config 5's 4.32 M prisms + 12.96 M tetrahedra.
`--mesh cylinder-quadratic`: the same mesh with quadratically curved wall elements (every type then carries
per-point metric terms); `--mesh hex`: periodic box of n^3 warped, randomly numbered hexahedra (NEXT-2), isentropic vortex.
"""
import argparse
import json
import sys
import time

import numpy as np


def totals(case, us):
    """sum over elements and points of omega |J| u_k (k = 0..4) and of the kinetic energy; FP64."""
    tot = np.zeros(6)
    for e, u in zip(case["eles"], us):
        w = e["wts"][:, None] * e["djac"]
        for k in range(5):
            tot[k] += (w * u[:, k, :]).sum()
        tot[5] += (w * 0.5 * (u[:, 1, :] ** 2 + u[:, 2, :] ** 2 + u[:, 3, :] ** 2) / u[:, 0, :]).sum()
    return tot


def adaptive(args, case, ctx, stream, ndof):
    import torch
    t1 = args.steps * args.dt
    ctx.rk_adaptive_run(0.0, 2 * args.dt, args.dt, args.adaptive, args.adaptive)    # warm-up: graph capture, registers
    ctx.set_state(case["u0"])
    tot0 = totals(case, ctx.get_state())
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    e0.record(stream)
    st, hist = ctx.rk_adaptive_run(0.0, t1, args.dt, args.adaptive, args.adaptive)
    e1.record(stream)
    e1.synchronize()
    sec = e0.elapsed_time(e1) * 1e-3
    natt = st["accepted"] + st["rejected"]
    tot1 = totals(case, ctx.get_state())
    acc = [h[0] for h in hist if h[2]]
    out = dict(mode="adaptive", tol=args.adaptive, t1=t1, dof=ndof, accepted=st["accepted"], rejected=st["rejected"],
               dt_min=min(acc), dt_max=max(acc), dt_next=st["dt_next"], ms_per_attempt=1e3 * sec / natt,
               gdof_rhs_per_s=ndof * 5 * natt / sec / 1e9, mass_drift=(tot1[0] - tot0[0]) / abs(tot0[0]),
               energy_drift=(tot1[4] - tot0[4]) / abs(tot0[4]))
    print(json.dumps(out))
    ctx.close()


def main():
    import torch
    from fr_inputs import cases
    from . import Context
    ap = argparse.ArgumentParser()
    ap.add_argument("--scale", type=int, default=2)
    ap.add_argument("--copies", type=int, default=1, help="disjoint copies of the mesh held as one case")
    ap.add_argument("--p", type=int, default=3)
    ap.add_argument("--prec", default="f32", choices=["f32", "f64"])
    ap.add_argument("--steps", type=int, default=1000)
    ap.add_argument("--dt", type=float, default=4e-6)
    ap.add_argument("--json", default=None)
    ap.add_argument("--mesh", default="cylinder", choices=["cylinder", "cylinder-quadratic", "hex"])
    ap.add_argument("--n", type=int, default=40, help="cells per direction of the hexahedral box")
    ap.add_argument("--adaptive", type=float, default=None, metavar="TOL",
                    help="step-size control (fr_rk_adaptive_run, atol = rtol = TOL) from t = 0 to steps * dt, starting at dt")
    args = ap.parse_args()
    if not torch.cuda.is_available():
        raise SystemExit("sustained needs a CUDA device (no CPU fallback)")
    t0 = time.time()
    if args.mesh == "hex":
        case = cases.config_hex(args.n, args.p, "ns", numbering="random", warp=0.1)
    else:
        case = cases.config3(p=args.p, ntheta=100 * args.scale, nz=15 * args.scale, seed=cases.SEEDS["c5"],
                             quadratic=args.mesh == "cylinder-quadratic")
    if args.copies > 1:
        case = cases.replicate(case, args.copies, amp=0.005, seed=cases.SEEDS["c5"], compact=True)
    ndof = cases.ndof(case)
    ne = {e["etype"]: e["neles"] for e in case["eles"]}
    print("mesh: %s elements, %d DOF, generated in %.0f s" % (ne, ndof, time.time() - t0), flush=True)
    stream = torch.cuda.Stream()
    ctx = Context(case, prec=args.prec, stepper="rk45", stream=stream.cuda_stream)
    ctx.set_state(case["u0"])
    free_b, total_b = torch.cuda.mem_get_info()
    hbm_gb = (total_b - free_b) / 1e9
    print("set-up done at %.0f s, device memory in use %.1f GB of %.1f" % (time.time() - t0, hbm_gb, total_b / 1e9), flush=True)
    if args.adaptive is not None:
        return adaptive(args, case, ctx, stream, ndof)
    marks = sorted(set(m for m in (0, 10, 100, 1000, args.steps) if m <= args.steps))
    what = ("hex box %d^3 warped: %d hex" % (args.n, ne.get("hex", 0)) if args.mesh == "hex" else
            "config3 generator x%d%s%s: %d pri + %d tet" % (args.scale, " quadratic" if args.mesh != "cylinder" else "",
                                                            ", %d disjoint copies" % args.copies if args.copies > 1 else "",
                                                            ne.get("pri", 0), ne.get("tet", 0)))
    out = dict(workload="%s, p=%d, NS, RK45[2R+], %s" % (what, args.p, args.prec), dof=ndof, dt=args.dt, hbm_in_use_gb=hbm_gb,
               checkpoints=[])
    done, gpu_s = 0, 0.0
    for m in marks:
        if m > done:
            e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            e0.record(stream)
            ctx.rk_run(args.dt, m - done)
            e1.record(stream)
            e1.synchronize()
            gpu_s += e0.elapsed_time(e1) * 1e-3
            done = m
        us = ctx.get_state()
        finite = bool(all(np.isfinite(u).all() for u in us))
        tot = totals(case, us) if finite else np.full(6, np.nan)
        out["checkpoints"].append(dict(step=m, finite=finite, mass=tot[0], mom=[tot[1], tot[2], tot[3]], energy=tot[4], kinetic=tot[5]))
        print("step %5d finite %s totals %s" % (m, finite, " ".join("%.10e" % x for x in tot)), flush=True)
        if not finite:
            break
    out["steps"] = done
    out["gdof_rhs_per_s"] = ndof * 5 * done / gpu_s / 1e9 if gpu_s > 0 else None
    out["ms_per_step"] = 1e3 * gpu_s / max(done, 1)
    c0 = out["checkpoints"][0]
    cl = out["checkpoints"][-1]
    out["relative_drift"] = dict(mass=(cl["mass"] - c0["mass"]) / abs(c0["mass"]), energy=(cl["energy"] - c0["energy"]) / abs(c0["energy"]),
                                 kinetic=(cl["kinetic"] - c0["kinetic"]) / abs(c0["kinetic"]))
    out["rhs_breakdown_ms"] = ctx.profile_rhs(reps=3)
    out["kernels_launched"] = ctx.launch_count()
    print(json.dumps(out))
    if args.json:
        with open(args.json, "w") as f:
            json.dump(out, f, indent=1)
    ctx.close()


if __name__ == "__main__":
    sys.exit(main())
