"""Pins for the CPU oracle (`oracle/fr_oracle.py`) -- what the theory fixes (BASELINE.json north_star):
free-stream preservation (T1), discrete conservation (T2), consistency order on a smooth manufactured field
against a sympy-derived analytic residual (T3 Euler, T4 Navier-Stokes), brute-force weak-DG agreement on
few-element meshes (T6), closed forms / textbook properties of the point-wise physics, BC invariants.
The paper prints no worked numerical example of an RHS, hence no golden values from it.
"""
import numpy as np
import pytest

from fr_inputs import cases, mesh as M, refelem as R, state
from oracle import fr_oracle as O
from oracle import weakdg as W
from util import conservation_defect, field_errors, oracle_rhs


# ---------------------------------------------------------------------------- T1 / T2
@pytest.mark.parametrize("system", ["euler", "ns"])
@pytest.mark.parametrize("p", [1, 2, 3])
def test_T1_freestream_and_T2_conservation_mixed(system, p):
    c = cases.config2(4, p, system, mu=0.05, numbering="random")
    fs = [state.freestream(e["xu"], v=(0.3, 0.2, -0.1)) for e in c["eles"]]
    d = oracle_rhs(c, fs)
    assert max(np.abs(x).max() for x in d) < 2e-11
    pert = state.perturb(fs, 0.05, 7, v=(0.3, 0.2, -0.1))
    d = oracle_rhs(c, pert)
    assert max(np.abs(x).max() for x in d) > 1e-2
    assert np.abs(conservation_defect(c, d)).max() < 1e-13


@pytest.mark.parametrize("system", ["euler", "ns"])
@pytest.mark.parametrize("p,warp", [(1, 0.0), (2, 0.0), (2, 0.12), (3, 0.12)])
def test_T1_T2_hexahedra(system, p, warp):
    """Hexahedra (NEXT-2): free-stream preservation and conservation, affine and warped (trilinear: the metric terms are of degree 2
    per direction, inside Q_p for p >= 2)."""
    c = cases.config_hex(3, p, system, mu=0.05, numbering="random", warp=warp)
    fs = [state.freestream(e["xu"], v=(0.3, 0.2, -0.1)) for e in c["eles"]]
    assert max(np.abs(x).max() for x in oracle_rhs(c, fs)) < 2e-11
    d = oracle_rhs(c, state.perturb(fs, 0.05, 7, v=(0.3, 0.2, -0.1)))
    assert max(np.abs(x).max() for x in d) > 1e-2
    assert np.abs(conservation_defect(c, d)).max() < 1e-13


@pytest.mark.parametrize("system", ["euler", "ns"])
@pytest.mark.parametrize("p", [2, 3, 4])
def test_T1_T2_quadratically_curved(system, p):
    """Quadratically curved elements (NEXT-1).  The metric terms S = |J| J^-1 of a P2 tetrahedron are of total
    degree 2, those of a P2 x P2 prism of degree 3 per direction: free-stream preservation holds to round-off once they lie in
    the element's polynomial space -- tetrahedra from p = 2, prisms from p = 3 (and visibly not at p = 2) -- while
    conservation is an algebraic identity at every p."""
    c = cases.config2(4, p, system, mu=0.05, numbering="random", curve=0.08)
    assert not c["eles"][0]["affine"] and not c["eles"][1]["affine"]
    fs = [state.freestream(e["xu"], v=(0.3, 0.2, -0.1)) for e in c["eles"]]
    r = oracle_rhs(c, fs)
    assert c["etypes"] == ["tet", "pri"]
    if p >= 3:
        assert max(np.abs(x).max() for x in r) < 5e-11
    else:
        # the error is born in the prisms; tetrahedra away from them stay clean
        assert np.abs(r[1]).max() > 1e-3
        clean = np.abs(r[0]).max(axis=(0, 1)) < 5e-11
        assert clean.sum() > 0.3 * clean.size
    d = oracle_rhs(c, state.perturb(fs, 0.05, 7, v=(0.3, 0.2, -0.1)))
    assert max(np.abs(x).max() for x in d) > 1e-2
    assert np.abs(conservation_defect(c, d)).max() < 1e-13


def test_T1_T2_config1():
    c = cases.config1()
    d = oracle_rhs(c)
    assert np.abs(conservation_defect(c, d)).max() < 1e-13
    fs = [state.freestream(e["xu"]) for e in c["eles"]]
    assert np.abs(oracle_rhs(c, fs)[0]).max() < 1e-13


@pytest.mark.parametrize("system", ["euler", "ns"])
def test_T1_wedge_prisms_and_farfield_boundary(system):
    # straight wedge prisms are non-affine: free-stream preservation needs p >= 2;
    # far field with u_L = u_inf returns u_inf, so everything away from the wall keeps dudt = 0
    nz, nl = 4, 4
    c = cases.config3(p=2, ntheta=16, nz=nz, nlayers=nl, nr=4, amp=0.0, numbering="natural", system=system)
    assert not c["eles"][1]["affine"]
    d = oracle_rhs(c)
    scale = 1.0 / c["eles"][1]["djac"].min() ** (1 / 3)   # ~ 1/h of the thinnest prism
    layer = (np.arange(c["eles"][1]["neles"]) // 2 // nz) % nl
    assert np.array_equal(np.unique(c["bcs"][0]["ele"]), np.nonzero(layer == 0)[0])
    # Euler: only wall prisms feel the wall.  NS: their gradients also reach the next layer through G_f.
    far = layer >= (1 if system == "euler" else 2)
    assert np.abs(d[1][:, :, far]).max() < 1e-11 * scale * 20
    assert np.abs(d[0]).max() < 1e-11 * scale * 20         # all tets (interior + far-field faces only)
    assert np.abs(d[1][:, :, layer == 0]).max() > 1.0      # the wall does act


def test_ns_rhs_is_affine_in_mu():
    c = cases.config2(4, 2, "ns", mu=0.0, state_kind="smooth")
    out = []
    for mu in (0.0, 0.01, 0.02):
        c["cfg"]["mu"] = mu
        out.append(oracle_rhs(c))
    for a, b, cc in zip(*out):
        assert np.abs((b - a) * 2 - (cc - a)).max() < 1e-11 * np.abs(cc).max()


# ---------------------------------------------------------------------------- point-wise physics
def _rand_states(n, seed):
    rng = np.random.default_rng(seed)
    rho = rng.uniform(0.5, 2.0, n)
    v = rng.uniform(-1, 1, (3, n))
    p = rng.uniform(0.5, 2.0, n)
    return state.prim_to_cons(rho, v, p), rho, v, p


def test_rusanov_textbook_properties():
    g = 1.4
    uL, rho, v, p = _rand_states(50, 1)
    uR = _rand_states(50, 2)[0]
    rng = np.random.default_rng(3)
    n = rng.standard_normal((3, 50))
    n /= np.linalg.norm(n, axis=0)
    # consistency F(u,u,n) = f(u).n ; f checked against the closed form of the Euler flux
    f = O.inviscid_flux(uL, g)
    vn = (v * n).sum(0)
    fn = np.stack([rho * vn, rho * v[0] * vn + p * n[0], rho * v[1] * vn + p * n[1], rho * v[2] * vn + p * n[2],
                   (uL[4] + p) * vn])
    assert np.abs(sum(f[i] * n[i] for i in range(3)) - fn).max() < 1e-14
    assert np.abs(O.rusanov(uL, uL, n, g) - fn).max() < 1e-14
    # conservation F(uL,uR,n) = -F(uR,uL,-n)
    assert np.abs(O.rusanov(uL, uR, n, g) + O.rusanov(uR, uL, -n, g)).max() < 1e-14
    # rotational invariance: rotating velocities and normal rotates the momentum flux
    Q, _ = np.linalg.qr(rng.standard_normal((3, 3)))
    rot = lambda u: np.concatenate([u[:1], Q @ u[1:4], u[4:]])
    assert np.abs(rot(O.rusanov(uL, uR, n, g)) - O.rusanov(rot(uL), rot(uR), Q @ n, g)).max() < 1e-13
    # dissipation coefficient is the largest |v.n| + c of the two sides
    lam = np.maximum(np.abs((uL[1:4] / uL[0] * n).sum(0)) + np.sqrt(g * p / rho),
                     O._normal_speed_plus_c(uR, n, g))
    central = 0.5 * sum((O.inviscid_flux(uL, g)[i] + O.inviscid_flux(uR, g)[i]) * n[i] for i in range(3))
    assert np.abs(O.rusanov(uL, uR, n, g) - central - 0.5 * lam * (uL - uR)).max() < 1e-13


def test_viscous_flux_closed_form_from_primitive_gradients():
    # build conserved gradients from chosen primitive gradients by the product rule, then compare with the
    # textbook stress tensor / Fourier heat flux evaluated directly from the primitive gradients
    g, mu, pr = 1.4, 0.37, 0.72
    u, rho, v, p = _rand_states(40, 4)
    rng = np.random.default_rng(5)
    drho, dv, dp = rng.standard_normal((3, 40)), rng.standard_normal((3, 3, 40)), rng.standard_normal((3, 40))
    q = np.zeros((3, 5, 40))
    for i in range(3):
        q[i, 0] = drho[i]
        for j in range(3):
            q[i, 1 + j] = drho[i] * v[j] + rho * dv[i, j]
        q[i, 4] = dp[i] / (g - 1) + 0.5 * drho[i] * (v ** 2).sum(0) + rho * (v * dv[i]).sum(0)
    f = O.viscous_flux(u, q, g, mu, pr)
    div = dv[0, 0] + dv[1, 1] + dv[2, 2]
    T = p / rho
    dT = (dp - T * drho) / rho
    kappa = mu * g / ((g - 1) * pr)                       # mu c_p / Pr with R = 1
    for i in range(3):
        tau = np.stack([mu * (dv[i, j] + dv[j, i] - (2 / 3) * div * (i == j)) for j in range(3)])
        assert np.abs(f[i, 0]).max() == 0
        assert np.abs(f[i, 1:4] - tau).max() < 1e-13
        assert np.abs(f[i, 4] - ((v * tau).sum(0) + kappa * dT[i])).max() < 1e-12
    # and the independent scalar implementation in the brute-force module agrees
    for k in range(5):
        fk = W.viscous_flux_pt(u[:, k], [q[i][:, k] for i in range(3)], g, mu, pr)
        assert np.abs(np.array(fk) - f[:, :, k]).max() < 1e-12


def test_boundary_ghost_state_invariants():
    g = 1.4
    rho_i, v_i, p_i = 1.0, np.array([1.0, 0.0, 0.0]), 1 / (1.4 * 0.04)
    uinf = state.prim_to_cons(np.full(30, rho_i), np.repeat(v_i[:, None], 30, 1), np.full(30, p_i))
    rng = np.random.default_rng(8)
    n = rng.standard_normal((3, 30))
    n /= np.linalg.norm(n, axis=0)
    # far field: u_L = u_inf  =>  u_b = u_inf for inflow and outflow normals
    ub = O.ghost_farfield(uinf, n, g, rho_i, v_i, p_i)
    assert np.abs(ub - uinf).max() < 1e-12
    # wall: with u_L at rest at the wall temperature the Riemann flux is pure pressure
    e_w = 2.3
    z = np.zeros(30)
    uL = np.stack([np.full(30, 1.7), z, z, z, 1.7 * e_w * np.ones(30)])
    ub, uw = O.ghost_wall(uL, e_w)
    assert np.abs(ub - uL).max() == 0 and np.abs(uw - uL).max() == 0
    F = O.rusanov(uL, ub, n, g)
    pw = (g - 1) * 1.7 * e_w
    assert np.abs(F[0]).max() < 1e-14 and np.abs(F[4]).max() < 1e-14 and np.abs(F[1:4] - pw * n).max() < 1e-13
    # moving fluid: ghost has reversed momentum, same density, wall internal energy + same kinetic energy
    uL2 = _rand_states(30, 9)[0]
    ub2, uw2 = O.ghost_wall(uL2, e_w)
    assert np.array_equal(ub2[1:4], -uL2[1:4]) and np.array_equal(ub2[0], uL2[0])
    ke = 0.5 * (uL2[1:4] ** 2).sum(0) / uL2[0]
    assert np.abs(ub2[4] - (uL2[0] * e_w + ke)).max() < 1e-14 and np.abs(uw2[1:4]).max() == 0


# ---------------------------------------------------------------------------- T6 brute force
def _weak_refs(case):
    refs = []
    for e in case["eles"]:
        o = R.operators(e["etype"], e["order"])
        refs.append(W.RefElement(e["etype"], e["order"], o["upts"], o["fpts"], o["fface"], o["fab"],
                                 R.verts(e["etype"]), o["faces"]))
    return refs


@pytest.mark.parametrize("kind,p,system", [("tets", 1, "euler"), ("tets", 2, "ns"), ("mixed", 2, "euler"),
                                           ("mixed", 2, "ns"), ("mixed", 3, "euler"), ("mixed1", 1, "ns")])
def test_T6_weak_dg_bruteforce(kind, p, system):
    if kind == "tets":
        m = M.box_tets(2, 1.0)
    elif kind == "mixed":
        m = M.box_mixed(2, 1.0)
    else:
        m = M.box_tets(1, 1.0)
    c = cases.build_case(m, p, system=system, mu=0.03 if system == "ns" else 0.0, by_coords=True)
    u0 = [state.smooth_periodic(e["xu"]) for e in c["eles"]]
    u0 = state.perturb(u0, 0.02, 12)
    ref = oracle_rhs(c, u0)
    refs = _weak_refs(c)
    # the operators themselves: M0 = interpolation, M3 = Mass^-1 B (lifting definition, reading R7)
    for e, r in zip(c["eles"], refs):
        assert np.abs(e["M0"] - r.interp).max() < 1e-11
        assert np.abs(e["M3"] - np.linalg.solve(r.mass, r.B)).max() < 1e-10
        o = R.operators(e["etype"], p)
        assert np.abs(o["fnorm"] - r.nhat).max() < 1e-14
    got = W.rhs(c["cfg"], refs, c["eles"], c["ifc"], u0)
    err, den = field_errors(got, ref)
    assert err.max() < 1e-10, err


# ---------------------------------------------------------------------------- T3 / T4 consistency order
def _analytic_residual(mu, pr=0.72, gamma=1.4, length=1.0):
    import sympy as sp
    x, y, z = sp.symbols("x y z")
    k = 2 * sp.pi / length
    rho = 1 + sp.Rational(1, 5) * sp.sin(k * (x + y + z))
    v = [sp.Rational(1, 2) + sp.Rational(1, 10) * sp.cos(k * (x - 2 * y)),
         sp.Rational(3, 10) + sp.Rational(1, 10) * sp.sin(k * (y + z)),
         sp.Rational(1, 5) + sp.Rational(1, 10) * sp.cos(k * (z - x))]
    p = 1 + sp.Rational(1, 10) * sp.cos(k * (x + y - z))
    X = [x, y, z]
    E = p / (gamma - 1) + rho * sum(c * c for c in v) / 2
    T = p / rho
    div = sum(sp.diff(v[i], X[i]) for i in range(3))
    tau = [[mu * (sp.diff(v[j], X[i]) + sp.diff(v[i], X[j]) - sp.Rational(2, 3) * div * (1 if i == j else 0))
            for j in range(3)] for i in range(3)]
    kappa = mu * gamma / ((gamma - 1) * pr)
    res = []
    flux = lambda i: [rho * v[i]] + [rho * v[i] * v[j] + (p if i == j else 0) - tau[i][j] for j in range(3)] + \
        [(E + p) * v[i] - sum(v[j] * tau[i][j] for j in range(3)) - kappa * sp.diff(T, X[i])]
    fl = [flux(i) for i in range(3)]
    for m in range(5):
        res.append(sp.lambdify(X, -sum(sp.diff(fl[i][m], X[i]) for i in range(3)), "numpy"))
    return res


@pytest.mark.parametrize("system,p,ns_,min_order", [("euler", 1, (8, 16), 0.75), ("euler", 2, (4, 8), 1.55),
                                                     ("euler", 3, (4, 8), 2.5), ("ns", 2, (4, 8), 0.6),
                                                     ("ns", 3, (4, 8), 1.5), ("hex-euler", 2, (6, 12), 1.5),
                                                     ("hex-ns", 3, (6, 12), 1.5), ("curved-euler", 3, (4, 8), 2.5),
                                                     ("curved-ns", 3, (4, 8), 1.3)])
def test_T3_T4_consistency_order(system, p, ns_, min_order):
    hexes = system.startswith("hex-")
    curve = 0.08 if system.startswith("curved-") else 0.0
    system = system.replace("hex-", "").replace("curved-", "")
    mu = 0.05 if system == "ns" else 0.0
    res = _analytic_residual(mu)
    errs = []
    for n in ns_:
        c = (cases.config_hex(n, p, system, mu=mu, state_kind="smooth", warp=0.1) if hexes
             else cases.config2(n, p, system, mu=mu, state_kind="smooth", curve=curve))
        d = oracle_rhs(c)
        num = np.zeros(5)
        for e, dd in zip(c["eles"], d):
            xu = e["xu"]
            for m in range(5):
                ex = res[m](xu[..., 0], xu[..., 1], xu[..., 2])
                w = e["wts"][:, None] * e["djac"]
                num[m] += (np.abs(w) * (dd[:, m, :] - ex) ** 2).sum()
        errs.append(np.sqrt(num))
    order = np.log2(errs[0] / errs[1])
    print(system, p, order)
    assert order.min() > min_order, (order, errs)
