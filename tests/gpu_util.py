"""Helpers for the GPU parity tests: torch owns the device memory, the library gets raw pointers."""
import copy

import numpy as np


def round_case_to_f32(case):
    """FP32 mode (reading R15): the library rounds every FP64 input once; the oracle consumes the same rounded
    values promoted back to FP64, so only arithmetic error is compared."""
    r = lambda a: np.asarray(a, dtype=np.float64).astype(np.float32).astype(np.float64)
    c = dict(case)
    c["cfg"] = dict(case["cfg"])
    for k in ("gamma", "mu", "prandtl", "ldg_beta", "ldg_tau"):
        c["cfg"][k] = float(np.float32(c["cfg"][k]))
    c["eles"] = []
    for e in case["eles"]:
        e2 = dict(e)
        for k in ("M0", "M132", "M3", "M460", "M6", "smats", "rcpdjac"):
            e2[k] = r(e[k])
        c["eles"].append(e2)
    c["ifc"] = dict(case["ifc"])
    for k in ("nl", "magl", "magr"):
        c["ifc"][k] = r(case["ifc"][k])
    c["bcs"] = []
    for b in case["bcs"]:
        b2 = dict(b)
        b2["n"], b2["mag"] = r(b["n"]), r(b["mag"])
        b2["params"] = [float(np.float32(x)) for x in b["params"]]
        c["bcs"].append(b2)
    if "u0" in case:
        c["u0"] = [r(u) for u in case["u0"]]
    return c


def to_device(ctx, us):
    import torch
    tdt = torch.float64 if ctx.prec == "f64" else torch.float32
    out = []
    for u, ld in zip(us, ctx.ld):
        nu, nv, ne = u.shape
        h = np.zeros((nu, nv, ld), dtype=ctx.dtype)
        h[:, :, :ne] = u
        # non-trivial garbage in the padding lanes: must be ignored on input
        h[:, :, ne:] = 7.0
        out.append(torch.from_numpy(h).to("cuda").to(tdt).contiguous())
    return out


def gpu_rhs(ctx, us):
    """fr_rhs through the C ABI; returns FP64 host arrays [nupts,5,neles] and the raw padded outputs."""
    import torch
    d_u = to_device(ctx, us)
    d_out = [torch.full_like(t, float("nan")) for t in d_u]
    ctx.rhs([t.data_ptr() for t in d_u], [t.data_ptr() for t in d_out])
    ctx.sync()
    torch.cuda.synchronize()
    raw = [t.cpu().numpy().astype(np.float64) for t in d_out]
    return [r[:, :, :u.shape[2]] for r, u in zip(raw, us)], raw


def subcase(case, seeds, rings=2):
    """Cut the `rings`-neighbourhood of the seed elements out of a case (same dict layout, elements renumbered).
    seeds: per element type an int array of element ids.  Returns (sub-case, per type the positions of the seeds in it).
    The right-hand side at an element depends on its neighbours (common flux) and, for Navier-Stokes, on their neighbours
    (their gradients need their common solution), so with rings = 2 the oracle evaluated on the sub-case reproduces the
    full-mesh values at the seeds exactly; flux points on the cut are simply left unpaired."""
    ifc = case["ifc"]
    nt = len(case["eles"])
    inset = [np.zeros(e["neles"], dtype=bool) for e in case["eles"]]
    for t in range(nt):
        inset[t][np.asarray(seeds[t], dtype=np.int64)] = True
    for _ in range(rings):
        lin = np.zeros(len(ifc["l_et"]), dtype=bool)
        rin = np.zeros(len(ifc["l_et"]), dtype=bool)
        for t in range(nt):
            ml, mr = ifc["l_et"] == t, ifc["r_et"] == t
            lin[ml] = inset[t][ifc["l_ele"][ml]]
            rin[mr] = inset[t][ifc["r_ele"][mr]]
        touch = lin | rin
        for t in range(nt):
            ml, mr = touch & (ifc["l_et"] == t), touch & (ifc["r_et"] == t)
            inset[t][ifc["l_ele"][ml]] = True
            inset[t][ifc["r_ele"][mr]] = True
    ids = [np.flatnonzero(m) for m in inset]
    remap = [np.full(len(m), -1, dtype=np.int64) for m in inset]
    for t in range(nt):
        remap[t][ids[t]] = np.arange(len(ids[t]))
    sub = dict(cfg=case["cfg"], etypes=case["etypes"], order=case["order"], eles=[], bcs=[])
    for t, e in enumerate(case["eles"]):
        e2 = dict(e)
        e2["neles"] = len(ids[t])
        for k in ("smats", "rcpdjac", "djac"):
            e2[k] = np.ascontiguousarray(e[k][..., ids[t]])
        e2["xu"] = np.ascontiguousarray(e["xu"][:, ids[t], :])
        sub["eles"].append(e2)
    keep = np.ones(len(ifc["l_et"]), dtype=bool)
    for t in range(nt):
        ml, mr = ifc["l_et"] == t, ifc["r_et"] == t
        keep[ml] &= inset[t][ifc["l_ele"][ml]]
        keep[mr] &= inset[t][ifc["r_ele"][mr]]
    s = {k: (v[keep] if v.ndim == 1 else v[:, keep]) for k, v in ifc.items()}
    for side in ("l", "r"):
        ne = s[side + "_ele"].copy()
        for t in range(nt):
            m = s[side + "_et"] == t
            ne[m] = remap[t][s[side + "_ele"][m]]
        s[side + "_ele"] = ne
    sub["ifc"] = s
    for b in case["bcs"]:
        kb = np.zeros(len(b["et"]), dtype=bool)
        for t in range(nt):
            m = b["et"] == t
            kb[m] = inset[t][b["ele"][m]]
        b2 = dict(b)
        for k in ("et", "fpt", "ele", "mag"):
            b2[k] = b[k][kb]
        b2["n"] = b["n"][:, kb]
        ne = b2["ele"].copy()
        for t in range(nt):
            m = b2["et"] == t
            ne[m] = remap[t][b2["ele"][m]]
        b2["ele"] = ne
        sub["bcs"].append(b2)
    sub["u0"] = [np.ascontiguousarray(u[:, :, ids[t]]) for t, u in enumerate(case["u0"])]
    return sub, [remap[t][np.asarray(seeds[t], dtype=np.int64)] for t in range(nt)]
