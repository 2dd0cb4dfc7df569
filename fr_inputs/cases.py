"""Assemble complete, seeded problem instances ("cases") for the configs of BASELINE.json.

A case carries exactly what `fr_setup` takes (include/frb200.h) and what the oracle takes
(oracle/fr_oracle.py `rhs`): operators, metric terms, flux-point pairs, boundary lists, parameters and
an initial state.  It contains no right-hand-side arithmetic.
"""
import numpy as np

from . import mesh as _mesh
from . import refelem, state

SEEDS = dict(c1=14090405, c2=14090406, c3=14090407, c4=14090408, c5=14090409)


def build_case(m, p, system="euler", gamma=state.GAMMA, mu=0.0, prandtl=0.72, ldg_beta=0.5, ldg_tau=0.1,
               bc_types=None, bc_params=None, by_coords=False):
    """mesh dict -> case dict(cfg, etypes, eles, ifc, bcs).  `bc_types`: {tag: 'wall'|'farfield'}."""
    eles, geo = [], {}
    for t in m["etypes"]:
        ops = refelem.operators(t, p)
        g = _mesh.geometry(t, p, m["xq"][t] if "xq" in m else m["xv"][t])
        geo[t] = g
        e = dict(etype=t, order=p, nupts=ops["nupts"], nfpts=ops["nfpts"], neles=m["xv"][t].shape[0],
                 affine=g["affine"], smats=g["smats"], rcpdjac=g["rcpdjac"], djac=g["djac"], xu=g["xu"],
                 wts=ops["wts"], fwts=ops["fwts"])
        for k in ("M0", "M132", "M3", "M460", "M6"):
            e[k] = ops[k]
        eles.append(e)
    if by_coords:
        ifc, bf = _mesh.connectivity_by_coords(m, p, geo)
    else:
        ifc, bf = _mesh.connectivity(m, p, geo)
    bcs = []
    for tag in sorted(bf):
        b = dict(bf[tag])
        b["type"] = bc_types[tag]
        b["params"] = list(bc_params[tag])
        bcs.append(b)
    cfg = dict(system=system, gamma=gamma, mu=mu, prandtl=prandtl, ldg_beta=ldg_beta, ldg_tau=ldg_tau)
    return dict(cfg=cfg, etypes=list(m["etypes"]), order=p, eles=eles, ifc=ifc, bcs=bcs, geo=geo, mesh=m)


def ndof(case):
    """DOF = sum over types of N_u * N_e (solution points; reading R22)."""
    return int(sum(e["nupts"] * e["neles"] for e in case["eles"]))


def config1(numbering="natural"):
    """BASELINE.json configs[0]: 384 Kuhn tets on the periodic cube [0,2pi]^3, p=2, Euler, FP64,
    freestream rho=1, v=(0.3,0,0), p=1/gamma + seeded 1 % perturbation (reading R17)."""
    m = _mesh.box_tets(4, 2 * np.pi, numbering=numbering, seed=SEEDS["c1"])
    case = build_case(m, 2, system="euler")
    fs = dict(rho=1.0, v=(0.3, 0.0, 0.0), p=1.0 / state.GAMMA)
    u0 = [state.freestream(e["xu"], **fs) for e in case["eles"]]
    case["u0"] = state.perturb(u0, 0.01, SEEDS["c1"], **fs)
    return case


def config2(n=16, p=3, system="ns", mu=1e-3, numbering="natural", state_kind="vortex", curve=0.0, ldg_beta=0.5, ldg_tau=0.1):
    """BASELINE.json configs[1]: periodic unit box, n^3 cells, lower half prisms / upper half tets
    (reading R18 for the counts), NS mu=1e-3 Pr=0.72, LDG beta=1/2 tau=0.1, isentropic vortex.
    curve > 0: the same mesh with quadratically curved elements."""
    m = _mesh.box_mixed(n, 1.0, numbering=numbering, seed=SEEDS["c2"], curve=curve)
    case = build_case(m, p, system=system, mu=mu if system == "ns" else 0.0, ldg_beta=ldg_beta, ldg_tau=ldg_tau)
    if state_kind == "vortex":
        case["u0"] = [state.isentropic_vortex(e["xu"]) for e in case["eles"]]
    else:
        case["u0"] = [state.smooth_periodic(e["xu"]) for e in case["eles"]]
    return case


def config_hex(n=8, p=3, system="ns", mu=1e-3, numbering="natural", warp=0.0, state_kind="vortex"):
    """Hexahedral periodic box (NEXT-2 of SURVEY 8(f): the paper's second mesh type), same physics as config 2."""
    m = _mesh.box_hex(n, 1.0, numbering=numbering, seed=SEEDS["c2"], warp=warp)
    case = build_case(m, p, system=system, mu=mu if system == "ns" else 0.0)
    if state_kind == "vortex":
        case["u0"] = [state.isentropic_vortex(e["xu"]) for e in case["eles"]]
    else:
        case["u0"] = [state.smooth_periodic(e["xu"]) for e in case["eles"]]
    return case


def config3(p=4, ntheta=100, nz=15, nlayers=40, nr=40, numbering="morton", system="ns", amp=0.005, seed=None, quadratic=False,
            mach=0.2, ldg_beta=0.5, ldg_tau=0.1):
    """BASELINE.json configs[2] (and [4] when scaled): cylinder-like O-mesh, NS at Re=3900, M=0.2
    (PAPER.md:86-94,116), wall T_w = T_inf, far field = freestream, seeded 0.5 % perturbation.
    `mach` > 1 drives the far-field boundary through its supersonic in- and outflow branches (test input only)."""
    seed = SEEDS["c3"] if seed is None else seed
    m = _mesh.cylinder_omesh(ntheta, nz, nlayers, nr, numbering=numbering, seed=seed, quadratic=quadratic)
    gamma = state.GAMMA
    fs = dict(rho=1.0, v=(1.0, 0.0, 0.0), p=1.0 / (gamma * mach * mach))
    e_w = fs["p"] / ((gamma - 1) * fs["rho"])
    case = build_case(m, p, system=system, mu=1.0 / 3900.0 if system == "ns" else 0.0, ldg_beta=ldg_beta, ldg_tau=ldg_tau,
                      bc_types={0: "wall", 1: "farfield"},
                      bc_params={0: [e_w], 1: [fs["rho"], *fs["v"], fs["p"]]})
    u0 = [state.freestream(e["xu"], **fs) for e in case["eles"]]
    case["u0"] = state.perturb(u0, amp, seed, **fs) if amp > 0 else u0
    case["freestream"] = fs
    return case


def replicate(case, copies, amp=None, seed=None, compact=False):
    """`copies` disjoint copies of a case as one case: copy k's elements of a type follow copy k-1's, its flux-point pairs and
    boundary lists follow copy k-1's with the element numbers shifted.  The copies do not touch; each keeps its own periodic
    span, wall and far field.  This is how the sustained run (BASELINE.json configs[4]) reaches sizes the host-side mesh
    generator cannot (ntheta x nz grows with the square of the scale): same element mix, operators, metric terms and
    connectivity structure per copy.  `amp`/`seed`: copy k > 0 gets its own seeded perturbation of the free stream
    (`case['freestream']` must be there); otherwise the initial state is tiled.  `compact=True` keeps one point of the
    metric terms of affine types (what fr_setup reads) and drops the coordinates, for very large cases."""
    K = int(copies)
    if K < 1:
        raise ValueError("copies must be >= 1")
    ne = [e["neles"] for e in case["eles"]]
    out = dict(cfg=dict(case["cfg"]), etypes=list(case["etypes"]), order=case["order"], copies=K)
    if "freestream" in case:
        out["freestream"] = case["freestream"]
    eles = []
    for e in case["eles"]:
        d = dict(e)
        d["neles"] = e["neles"] * K
        cut = slice(0, 1) if (compact and e["affine"]) else slice(None)
        d["smats"] = np.tile(e["smats"][:, :, cut, :], (1, 1, 1, K))
        d["rcpdjac"] = np.tile(e["rcpdjac"][cut, :], (1, K))
        d["djac"] = np.tile(e["djac"][cut, :], (1, K))
        d["xu"] = None if compact else np.tile(e["xu"], (1, K, 1))
        eles.append(d)
    out["eles"] = eles
    nea = np.asarray(ne, dtype=np.int64)

    def shifted(et, ele):
        return (ele[None, :] + np.arange(K, dtype=np.int64)[:, None] * nea[et][None, :]).reshape(-1)

    ifc = case["ifc"]
    o = {}
    for side in ("l", "r"):
        o[side + "_et"] = np.tile(ifc[side + "_et"], K)
        o[side + "_fpt"] = np.tile(ifc[side + "_fpt"], K)
        o[side + "_ele"] = shifted(ifc[side + "_et"], ifc[side + "_ele"])
    o["nl"] = np.tile(ifc["nl"], (1, K))
    o["magl"] = np.tile(ifc["magl"], K)
    o["magr"] = np.tile(ifc["magr"], K)
    out["ifc"] = o
    bcs = []
    for b in case["bcs"]:
        d = dict(b)
        d["et"] = np.tile(b["et"], K)
        d["fpt"] = np.tile(b["fpt"], K)
        d["ele"] = shifted(b["et"], b["ele"])
        d["n"] = np.tile(b["n"], (1, K))
        d["mag"] = np.tile(b["mag"], K)
        bcs.append(d)
    out["bcs"] = bcs
    if "u0" in case:
        u0 = [np.tile(u, (1, 1, K)) for u in case["u0"]]
        if amp is not None and K > 1:
            fs = case["freestream"]
            for k in range(1, K):
                base = [state.freestream(e["xu"], **fs) for e in case["eles"]]
                pk = state.perturb(base, amp, (SEEDS["c5"] if seed is None else seed) + k, **fs)
                for u, p_, n in zip(u0, pk, ne):
                    u[:, :, k * n:(k + 1) * n] = p_
        out["u0"] = u0
    return out
