"""Second set of pins for the CPU oracle (VERDICT r01 "What's weak" 1): the branches and conventions of `oracle/fr_oracle.py`
that the first set never exercised.

  * `ghost_farfield` (PAPER.md:94 names the type; formulas = SURVEY A.8, reading R11): all four branch combinations, checked
    against what characteristic theory fixes -- supersonic inflow returns u_inf whatever the interior state, supersonic outflow
    returns the interior state whatever u_inf, and in the subsonic cases the Riemann invariants, the entropy and the tangential
    velocity RECOMPUTED FROM u_b equal the ones carried by the corresponding characteristics.
  * LDG constants (reading R9): conservation (T2) and the brute-force weak-DG form (T6) for beta in {0, -1/2, 0.3} and
    tau in {0, 1}; the PAIRING of the switches -- the common solution takes (1/2 - beta, 1/2 + beta) and the common viscous flux
    the opposite weights -- is what makes the discrete diffusion operator self-adjoint and negative semi-definite in the mass
    inner product (div = -grad^T), and the SIGN of the penalty tau (u_L - u_R) is what makes it remove jump energy.
  * `rk4_step` / `rk45_step`: convergence slope on the non-linear ODE u' = -u^2 (exact solution 1/(1+t)), which sees the
    non-linear order conditions, and the two-register recurrence against the scheme's Butcher tableau written out stage by
    stage (the tableau itself is pinned by the exact order conditions in test_rk.py).
"""
from fractions import Fraction

import numpy as np
import pytest

from fr_inputs import cases, mesh as M, refelem as R, state
from oracle import fr_oracle as O
from oracle import weakdg as W
from util import conservation_defect, field_errors, oracle_rhs

G = 1.4


def _prim(u):
    rho = u[0]
    v = u[1:4] / rho
    p = (G - 1) * (u[4] - 0.5 * rho * (v ** 2).sum(0))
    return rho, v, p


def _states(n, seed, mach):
    """n random states with |v| = mach * c, random directions."""
    rng = np.random.default_rng(seed)
    rho = rng.uniform(0.7, 1.4, n)
    p = rng.uniform(0.8, 1.6, n)
    d = rng.standard_normal((3, n))
    d /= np.linalg.norm(d, axis=0)
    c = np.sqrt(G * p / rho)
    return state.prim_to_cons(rho, mach * c * d, p)


def _unit(n, seed):
    x = np.random.default_rng(seed).standard_normal((3, n))
    return x / np.linalg.norm(x, axis=0)


# ---------------------------------------------------------------------------- far-field ghost state, four branches
def test_farfield_supersonic_inflow_returns_freestream():
    n = 64
    rho_i, p_i = 1.1, 0.9
    c_i = np.sqrt(G * p_i / rho_i)
    nrm = _unit(n, 1)
    for mach in (1.01, 1.5, 3.0):                     # v_n,inf = -mach c_inf <= -c_inf: both characteristics come from outside
        rng = np.random.default_rng(2)
        t = np.cross(nrm.T, rng.standard_normal((n, 3))).T * 0.3          # tangential part, any size
        for k in range(n):
            v_i = -mach * c_i * nrm[:, k] + t[:, k]
            # interior: anything that is not supersonic outflow (v_n < c)
            uL = _states(1, 10 + k, 0.6)
            ub = O.ghost_farfield(uL, nrm[:, k:k + 1], G, rho_i, v_i, p_i)
            uinf = state.prim_to_cons(np.array([rho_i]), v_i[:, None], np.array([p_i]))
            assert np.abs(ub - uinf).max() < 1e-12 * np.abs(uinf).max(), (mach, k)


def test_farfield_supersonic_outflow_returns_interior_state():
    n = 64
    nrm = _unit(n, 3)
    rng = np.random.default_rng(4)
    rho = rng.uniform(0.7, 1.4, n)
    p = rng.uniform(0.8, 1.6, n)
    c = np.sqrt(G * p / rho)
    for mach in (1.01, 1.7):                          # v_n,L = mach c_L >= c_L: both characteristics leave
        t = np.cross(nrm.T, rng.standard_normal((n, 3))).T * 0.4
        v = mach * c * nrm + t
        uL = state.prim_to_cons(rho, v, p)
        # far field: anything that is not supersonic inflow for this normal
        for v_inf in (np.array([0.1, -0.2, 0.05]), np.array([0.0, 0.0, 0.0])):
            ub = O.ghost_farfield(uL, nrm, G, 0.9, v_inf, 1.2)
            assert np.abs(ub - uL).max() < 1e-12 * np.abs(uL).max()


@pytest.mark.parametrize("case", ["sub_in", "sub_out", "mixed"])
def test_farfield_subsonic_branches_carry_the_right_invariants(case):
    n = 200
    nrm = _unit(n, 5)
    rho_i, p_i = 1.0, 1.2
    c_i = np.sqrt(G * p_i / rho_i)
    rng = np.random.default_rng(6)
    if case == "sub_in":        # |v_n| subsonic on both sides, far field blows in
        v_i = (-0.4 * c_i * nrm + np.cross(nrm.T, rng.standard_normal((n, 3))).T * 0.2)
        uL = _states(n, 7, 0.3)
    elif case == "sub_out":
        v_i = (0.4 * c_i * nrm + np.cross(nrm.T, rng.standard_normal((n, 3))).T * 0.2)
        uL = _states(n, 8, 0.3)
    else:                       # far field supersonic inflow AND interior supersonic outflow: R+ from outside, R- from inside
        v_i = -1.4 * c_i * nrm
        rho = rng.uniform(0.7, 1.4, n)
        p = rng.uniform(4.0, 6.0, n)
        uL = state.prim_to_cons(rho, 1.3 * np.sqrt(G * p / rho) * nrm, p)
    rL, vL, pL = _prim(uL)
    cL = np.sqrt(G * pL / rL)
    vnL = (vL * nrm).sum(0)
    ub = np.empty_like(uL)
    for k in range(n):          # per-point free stream (the routine takes one v_inf)
        ub[:, k:k + 1] = O.ghost_farfield(uL[:, k:k + 1], nrm[:, k:k + 1], G, rho_i, v_i[:, k], p_i)
    rb, vb, pb = _prim(ub)
    cb = np.sqrt(G * pb / rb)
    vnb = (vb * nrm).sum(0)
    vn_i = (v_i * nrm).sum(0)
    Rp_b, Rm_b = vnb + 2 * cb / (G - 1), vnb - 2 * cb / (G - 1)
    if case == "mixed":
        assert np.all(vn_i <= -c_i) and np.all(vnL >= cL)
        assert np.abs(Rp_b - (vn_i + 2 * c_i / (G - 1))).max() < 1e-11
        assert np.abs(Rm_b - (vnL - 2 * cL / (G - 1))).max() < 1e-11
        return
    assert np.all(np.abs(vn_i) < c_i) and np.all(np.abs(vnL) < cL)
    # outgoing invariant from the interior, incoming from the far field
    assert np.abs(Rp_b - (vnL + 2 * cL / (G - 1))).max() < 1e-11
    assert np.abs(Rm_b - (vn_i - 2 * c_i / (G - 1))).max() < 1e-11
    inflow = vnb < 0
    assert inflow.any() if case == "sub_in" else (~inflow).any()     # both branches of the entropy / velocity choice get exercised
    s_b = pb / rb ** G
    s_ref = np.where(inflow, p_i / rho_i ** G, pL / rL ** G)
    assert np.abs(s_b / s_ref - 1).max() < 1e-12
    # tangential velocity: the far field's on inflow, the interior's on outflow
    vt_b = vb - vnb * nrm
    vt_ref = np.where(inflow, v_i - vn_i * nrm, vL - vnL * nrm)
    assert np.abs(vt_b - vt_ref).max() < 1e-12


# ---------------------------------------------------------------------------- LDG constants
@pytest.mark.parametrize("beta,tau", [(0.0, 0.0), (-0.5, 1.0), (0.3, 0.1), (0.3, 1.0), (0.5, 0.0)])
def test_T2_conservation_for_other_ldg_constants(beta, tau):
    c = cases.config2(4, 2, "ns", mu=0.05, numbering="random", ldg_beta=beta, ldg_tau=tau)
    fs = [state.freestream(e["xu"], v=(0.3, 0.2, -0.1)) for e in c["eles"]]
    assert max(np.abs(x).max() for x in oracle_rhs(c, fs)) < 2e-11
    d = oracle_rhs(c, state.perturb(fs, 0.05, 7, v=(0.3, 0.2, -0.1)))
    assert np.abs(conservation_defect(c, d)).max() < 1e-13


def _weak_refs(case):
    refs = []
    for e in case["eles"]:
        o = R.operators(e["etype"], e["order"])
        refs.append(W.RefElement(e["etype"], e["order"], o["upts"], o["fpts"], o["fface"], o["fab"], R.verts(e["etype"]), o["faces"]))
    return refs


@pytest.mark.parametrize("beta,tau", [(0.0, 1.0), (-0.5, 0.0), (0.3, 0.1)])
def test_T6_weak_dg_for_other_ldg_constants(beta, tau):
    m = M.box_mixed(2, 1.0)
    c = cases.build_case(m, 2, system="ns", mu=0.03, by_coords=True, ldg_beta=beta, ldg_tau=tau)
    u0 = state.perturb([state.smooth_periodic(e["xu"]) for e in c["eles"]], 0.02, 12)
    got = W.rhs(c["cfg"], _weak_refs(c), c["eles"], c["ifc"], u0)
    err, _ = field_errors(got, oracle_rhs(c, u0))
    assert err.max() < 1e-10, err


def _mass_inner(case, refs, a, b):
    """sum over types and elements of a^T (|J| Mass) b, per variable; affine elements (|J| constant per element)."""
    out = np.zeros(5)
    for e, r, x, y in zip(case["eles"], refs, a, b):
        assert e["affine"]
        out += np.einsum("rve,rn,nve,e->v", x, r.mass, y, e["djac"][0])
    return out


def _energy_field(case, seed, amp=1e-3):
    """rho = 1, v = 0, E = E0 + amp * random: with it the energy equation's viscous part is a linear diffusion of E."""
    rng = np.random.default_rng(seed)
    us, phis = [], []
    for e in case["eles"]:
        u = state.freestream(e["xu"], rho=1.0, v=(0.0, 0.0, 0.0), p=1.0)
        phi = rng.uniform(-1, 1, (u.shape[0], u.shape[2]))
        u[:, 4, :] += amp * phi
        us.append(u)
        phis.append(phi)
    return us, phis


@pytest.mark.parametrize("beta", [0.3, -0.5, 0.5, 0.0])
def test_ldg_switch_pairing_makes_diffusion_self_adjoint_and_dissipative(beta):
    """With rho = 1 and v = 0 the viscous part of the energy equation is dE/dt = kappa' L E with L the scheme's discrete
    Laplacian.  LDG's opposite switches (C: (1/2-beta, 1/2+beta); viscous flux: (1/2+beta, 1/2-beta)) give div = -grad^T in the
    mass inner product, hence <phi, L psi> = <psi, L phi> and <phi, L phi> <= 0 for ANY beta; with the same switch on both
    (a transposition slip) L is not symmetric unless beta = 0."""
    mu, amp = 0.05, 1e-3

    def L(case0, case1, us):
        # viscous part alone: RHS is affine in mu (test_ns_rhs_is_affine_in_mu), the tau penalty is the same in both
        return [a - b for a, b in zip(oracle_rhs(case1, us), oracle_rhs(case0, us))]

    m = M.box_mixed(2, 1.0)
    c0 = cases.build_case(m, 2, system="ns", mu=0.0, by_coords=True, ldg_beta=beta, ldg_tau=0.0)
    c1 = cases.build_case(m, 2, system="ns", mu=mu, by_coords=True, ldg_beta=beta, ldg_tau=0.0)
    refs = _weak_refs(c1)
    (ua, pa), (ub, pb) = _energy_field(c1, 21, amp), _energy_field(c1, 22, amp)
    La, Lb = L(c0, c1, ua), L(c0, c1, ub)

    def as_state(phis):
        out = []
        for ph in phis:
            s = np.zeros((ph.shape[0], 5, ph.shape[1]))
            s[:, 4, :] = ph
            out.append(s)
        return out

    sa, sb = as_state(pa), as_state(pb)
    ab = _mass_inner(c1, refs, sa, Lb)[4]
    ba = _mass_inner(c1, refs, sb, La)[4]
    aa = _mass_inner(c1, refs, sa, La)[4]
    bb = _mass_inner(c1, refs, sb, Lb)[4]
    scale = max(abs(aa), abs(bb))
    assert scale > 0
    assert aa < 0 and bb < 0                                    # diffusion removes energy
    assert abs(ab - ba) < 1e-9 * scale, (ab, ba, scale)          # self-adjoint
    # the switch direction matters: the mirrored scheme (-beta, still paired) is self-adjoint too but a different operator
    if beta != 0.0:
        cw0 = cases.build_case(m, 2, system="ns", mu=0.0, by_coords=True, ldg_beta=-beta, ldg_tau=0.0)
        cw1 = cases.build_case(m, 2, system="ns", mu=mu, by_coords=True, ldg_beta=-beta, ldg_tau=0.0)
        Lw = L(cw0, cw1, ua)
        diff = max(np.abs(x - y).max() for x, y in zip(Lw, La))
        assert diff > 1e-3 * max(np.abs(x).max() for x in La)


def test_ldg_wrong_pairing_would_fail_the_symmetry_pin():
    """The symmetry pin above has teeth: assemble the diffusion operator from the oracle's own pieces with the viscous-flux
    switch deliberately set equal to the common-solution switch (both (1/2 - beta) on L) and see the symmetry break."""
    beta, mu = 0.3, 0.05
    m = M.box_mixed(2, 1.0)
    c = cases.build_case(m, 2, system="ns", mu=mu, by_coords=True, ldg_beta=beta, ldg_tau=0.0)
    refs = _weak_refs(c)
    eles, ifc = c["eles"], c["ifc"]
    L_ = (ifc["l_et"], ifc["l_fpt"], ifc["l_ele"])
    R_ = (ifc["r_et"], ifc["r_fpt"], ifc["r_ele"])

    def lap(phis, flux_beta):
        """scalar diffusion d phi/dt = div grad phi through the FR operators, C switch = beta, flux switch = flux_beta"""
        uf = [O._apply(e["M0"], p[:, None, :]) for e, p in zip(eles, phis)]
        uL, uR = O._gather(uf, *L_), O._gather(uf, *R_)
        cf = [np.zeros_like(a) for a in uf]
        C = (0.5 - beta) * uL + (0.5 + beta) * uR
        O._scatter(cf, *L_, C)
        O._scatter(cf, *R_, C)
        grads, gf = [], []
        for e, p, cc in zip(eles, phis, cf):
            nu = p.shape[0]
            gt = (O._apply(e["M460"], p[:, None, :]) + O._apply(e["M6"], cc)).reshape((3, nu, 1, -1))
            S, rj = e["smats"], e["rcpdjac"]
            g = np.stack([rj[:, None, :] * sum(S[a, i][:, None, :] * gt[a] for a in range(3)) for i in range(3)])
            grads.append(g)
            gf.append(np.stack([O._apply(e["M0"], g[i]) for i in range(3)]))
        qL = np.stack([O._gather([g[i] for g in gf], *L_) for i in range(3)])
        qR = np.stack([O._gather([g[i] for g in gf], *R_) for i in range(3)])
        n = ifc["nl"]
        Fc = -sum(((0.5 + flux_beta) * qL[i] + (0.5 - flux_beta) * qR[i]) * n[i] for i in range(3))
        d = [np.zeros_like(a) for a in uf]
        O._scatter(d, *L_, ifc["magl"] * Fc)
        O._scatter(d, *R_, -ifc["magr"] * Fc)
        out = []
        for e, g, dd in zip(eles, grads, d):
            nu = e["M132"].shape[0]
            S = e["smats"]
            ft = np.stack([sum(S[a, i][:, None, :] * (-g[i]) for i in range(3)) for a in range(3)])
            r = O._apply(e["M132"], ft.reshape(3 * nu, 1, -1)) + O._apply(e["M3"], dd)
            out.append((-r * e["rcpdjac"][:, None, :])[:, 0, :])
        return out

    rng = np.random.default_rng(5)
    pa = [rng.uniform(-1, 1, (e["nupts"], e["neles"])) for e in eles]
    pb = [rng.uniform(-1, 1, (e["nupts"], e["neles"])) for e in eles]

    def inner(a, b):
        return sum(np.einsum("re,rn,ne,e->", x, r.mass, y, e["djac"][0]) for e, r, x, y in zip(eles, refs, a, b))

    for fb, symmetric in ((beta, True), (-beta, False)):
        La, Lb = lap(pa, fb), lap(pb, fb)
        asym = abs(inner(pa, Lb) - inner(pb, La)) / abs(inner(pa, La))
        assert (asym < 1e-10) == symmetric, (fb, asym)


def test_penalty_sign_removes_jump_energy():
    """P(u) = RHS(tau = 1) - RHS(tau = 0) at mu = 0 is the penalty term alone, linear in u: with + tau (u_L - u_R) in the common
    flux, <u_k, P u_k> = -tau sum_faces int [u_k]^2 < 0 in the mass inner product, for every variable; with the other sign it
    would be positive."""
    m = M.box_mixed(2, 1.0)
    c0 = cases.build_case(m, 2, system="ns", mu=0.0, by_coords=True, ldg_beta=0.3, ldg_tau=0.0)
    c1 = cases.build_case(m, 2, system="ns", mu=0.0, by_coords=True, ldg_beta=0.3, ldg_tau=1.0)
    refs = _weak_refs(c1)
    u = state.perturb([state.smooth_periodic(e["xu"]) for e in c1["eles"]], 0.05, 3)
    P = [a - b for a, b in zip(oracle_rhs(c1, u), oracle_rhs(c0, u))]
    e_k = _mass_inner(c1, refs, u, P)
    assert np.all(e_k < 0), e_k
    # size: -tau * sum over faces of int [u_k]^2, estimated here with the flux points' own interpolatory face weights (exact to
    # degree p only, the integrand has degree 2p: an estimate, good to ~10 %)
    ifc = c1["ifc"]
    uf = [O._apply(e["M0"], x) for e, x in zip(c1["eles"], u)]
    uL = O._gather(uf, ifc["l_et"], ifc["l_fpt"], ifc["l_ele"])
    uR = O._gather(uf, ifc["r_et"], ifc["r_fpt"], ifc["r_ele"])
    wl = np.empty(len(ifc["l_et"]))
    for t, e in enumerate(c1["eles"]):
        mk = ifc["l_et"] == t
        wl[mk] = e["fwts"][ifc["l_fpt"][mk]]
    want = -(wl * ifc["magl"] * (uL - uR) ** 2).sum(axis=1)
    assert np.abs(e_k / want - 1).max() < 0.2, (e_k, want)


# ---------------------------------------------------------------------------- steppers on a non-linear ODE
def test_rk_slopes_on_nonlinear_ode():
    f = lambda us: [-u * u for u in us]
    exact = 1.0 / (1.0 + 1.0)
    for step, order in ((O.euler_step, 1), (O.rk4_step, 4), (O.rk45_step, 4)):
        errs = []
        for n in (4, 8, 16, 32):
            u = [np.array([1.0])]
            for _ in range(n):
                u = step(f, u, 1.0 / n)
            errs.append(abs(u[0][0] - exact))
        slopes = np.log2(np.array(errs[:-1]) / np.array(errs[1:]))
        assert np.all(slopes[1:] > order - 0.25) and np.all(slopes[1:] < order + 0.7), (step.__name__, slopes)


def test_rk45_two_register_form_equals_its_butcher_tableau():
    """The 2R recurrence X <- X + dt b_i K, Y <- X + dt (a_i - b_i) K must be the explicit Runge-Kutta scheme with
    A[i][i-1] = a_{i-1}, A[i][j] = b_j (j < i-1), weights b -- evaluated here stage by stage from the tableau
    on a non-linear system; the tableau's own order conditions are checked exactly in test_rk.py."""
    a = [float(Fraction(n, d)) for n, d in O.RK45_A_FRAC]
    b = [float(Fraction(n, d)) for n, d in O.RK45_B_FRAC]
    A = np.zeros((5, 5))
    for i in range(1, 5):
        for j in range(i):
            A[i, j] = a[j] if j == i - 1 else b[j]
    f1 = lambda u: np.array([-u[0] * u[1], u[0] * u[0] - 0.3 * u[1], np.sin(u[2]) + u[0]])
    u0 = np.array([0.7, -0.4, 0.2])
    dt = 0.37
    K = []
    for i in range(5):
        K.append(f1(u0 + dt * sum(A[i, j] * K[j] for j in range(i))))
    want = u0 + dt * sum(b[i] * K[i] for i in range(5))
    got = O.rk45_step(lambda us: [f1(us[0])], [u0.copy()], dt)[0]
    assert np.abs(got - want).max() < 1e-15
    got2, E = O.rk45_step_with_error(lambda us: [f1(us[0])], [u0.copy()], dt)
    assert np.abs(got2[0] - want).max() < 1e-15
    bh = [float(Fraction(n, d)) for n, d in O.RK45_BHAT_FRAC]
    assert np.abs(E[0] - dt * sum((b[i] - bh[i]) * K[i] for i in range(5))).max() < 1e-15
    # classical RK4 against its tableau as well
    k1 = f1(u0)
    k2 = f1(u0 + 0.5 * dt * k1)
    k3 = f1(u0 + 0.5 * dt * k2)
    k4 = f1(u0 + dt * k3)
    assert np.abs(O.rk4_step(lambda us: [f1(us[0])], [u0.copy()], dt)[0] - (u0 + dt / 6 * (k1 + 2 * k2 + 2 * k3 + k4))).max() < 1e-15
