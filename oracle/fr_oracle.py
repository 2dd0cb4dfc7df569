"""CPU ORACLE -- TEST INFRASTRUCTURE, NOT PRODUCT CODE.

Plain FP64 numpy evaluation of the flux-reconstruction right-hand side and Runge-Kutta steps that
the CUDA library (`include/frb200.h`) must reproduce.  Only `tests/`, `__graft_entry__.smoke()` and
the `cpu_baseline` / `--impl reference` legs of `bench.py` may import this package; it shares no
code with `paper_1409_0405_b200/` and imports nothing from it.

What the paper fixes (PAPER.md = /root/reference/PAPER.md):
  * every operator application is `C <- c1*A*B + c2*C` with a constant operator A and row-major
    state matrices B, C (eq. 1)  -> the `@` products below, nothing blocked or fused;
  * all other work is point-wise at a single solution / flux point;
  * compressible Navier-Stokes, constant viscosity, DG scheme (through the operators), Rusanov
    Riemann solver, RK45[2R+]; Euler / RK4 also exist (Table 1);
  * boundary-condition TYPES of the cylinder case.
Everything the paper is silent on (formulas of the FR factorisation, Rusanov wave speed, LDG
constants, viscous flux form, BC formulas, RK coefficients) follows the readings R4, R8-R12 listed in
DESIGN.md and is pinned by the theory tests in `tests/`
(free-stream preservation, conservation, consistency order, weak-DG brute force, closed forms).
Parity unpinned by the paper itself: the numerical values of beta, tau and the far-field / wall
ghost-state formulas (conventions; pinned only through their invariants).

Arrays: state of one element type U [N_u, 5, N_e] (variables rho, rho*v_x, rho*v_y, rho*v_z, E);
flux-point arrays [N_f, 5, N_e]; gradients [3, N_u, 5, N_e].  Steps are numbered as in SURVEY 8(c).
"""
import numpy as np

# ----------------------------------------------------------------------------- point-wise physics


def inviscid_flux(u, gamma):
    """f^inv_i: u [5, ...] -> f [3, 5, ...]; ideal gas p = (gamma-1)(E - rho|v|^2/2)."""
    rho, E = u[0], u[4]
    v = u[1:4] / rho
    p = (gamma - 1.0) * (E - 0.5 * rho * (v[0] ** 2 + v[1] ** 2 + v[2] ** 2))
    f = np.empty((3,) + u.shape)
    for i in range(3):
        f[i, 0] = rho * v[i]
        for j in range(3):
            f[i, 1 + j] = rho * v[i] * v[j] + (p if i == j else 0.0)
        f[i, 4] = (E + p) * v[i]
    return f


def viscous_flux(u, q, gamma, mu, prandtl):
    """f^visc_i (reading R10): u [5,...], q [3,5,...] = d u / d x_i -> f [3,5,...].
    Newtonian, Stokes hypothesis, constant mu, Fourier heat flux kappa = mu c_p / Pr."""
    rho, E = u[0], u[4]
    v = u[1:4] / rho
    dv = np.empty((3, 3) + rho.shape)                      # dv[i, j] = d_i v_j
    for i in range(3):
        for j in range(3):
            dv[i, j] = (q[i, 1 + j] - v[j] * q[i, 0]) / rho
    div = dv[0, 0] + dv[1, 1] + dv[2, 2]
    f = np.zeros((3,) + u.shape)
    for i in range(3):
        # rho d_i e = d_i E - (E/rho) d_i rho - rho sum_j v_j d_i v_j
        rho_de = q[i, 4] - (E / rho) * q[i, 0] - rho * (v[0] * dv[i, 0] + v[1] * dv[i, 1] + v[2] * dv[i, 2])
        work = 0.0
        for j in range(3):
            tau = mu * (dv[i, j] + dv[j, i] - (2.0 / 3.0) * div * (1.0 if i == j else 0.0))
            f[i, 1 + j] = tau
            work = work + v[j] * tau
        f[i, 4] = work + (mu * gamma / prandtl) * rho_de / rho
    return f


def _normal_speed_plus_c(u, n, gamma):
    rho = u[0]
    v = u[1:4] / rho
    p = (gamma - 1.0) * (u[4] - 0.5 * rho * (v[0] ** 2 + v[1] ** 2 + v[2] ** 2))
    return np.abs(v[0] * n[0] + v[1] * n[1] + v[2] * n[2]) + np.sqrt(gamma * p / rho)


def rusanov(uL, uR, n, gamma):
    """Rusanov / local Lax-Friedrichs normal flux (wave speed = reading R8):
    F = 1/2 (f(uL)+f(uR)).n + 1/2 lambda (uL-uR), lambda = max(|vL.n|+cL, |vR.n|+cR)."""
    fL, fR = inviscid_flux(uL, gamma), inviscid_flux(uR, gamma)
    lam = np.maximum(_normal_speed_plus_c(uL, n, gamma), _normal_speed_plus_c(uR, n, gamma))
    fn = 0.5 * sum((fL[i] + fR[i]) * n[i] for i in range(3))
    return fn + 0.5 * lam * (uL - uR)


def ghost_wall(uL, e_w):
    """No-slip isothermal wall (formulas = SURVEY A.8, reading R11).
    Returns (u_b for the inviscid Riemann problem, u_w wall state for the viscous part)."""
    rho = uL[0]
    ke = 0.5 * (uL[1] ** 2 + uL[2] ** 2 + uL[3] ** 2) / rho
    ub = np.stack([rho, -uL[1], -uL[2], -uL[3], rho * e_w + ke])
    z = np.zeros_like(rho)
    uw = np.stack([rho, z, z, z, rho * e_w])
    return ub, uw


def ghost_farfield(uL, n, gamma, rho_inf, v_inf, p_inf):
    """Riemann-invariant far field (formulas = SURVEY A.8, reading R11)."""
    g1 = gamma - 1.0
    rho = uL[0]
    v = uL[1:4] / rho
    p = g1 * (uL[4] - 0.5 * rho * (v[0] ** 2 + v[1] ** 2 + v[2] ** 2))
    c = np.sqrt(gamma * p / rho)
    vn = v[0] * n[0] + v[1] * n[1] + v[2] * n[2]
    c_inf = np.sqrt(gamma * p_inf / rho_inf)
    vn_inf = v_inf[0] * n[0] + v_inf[1] * n[1] + v_inf[2] * n[2]
    Rp = np.where(vn_inf <= -c_inf, vn_inf + 2 * c_inf / g1, vn + 2 * c / g1)
    Rm = np.where(vn >= c, vn - 2 * c / g1, vn_inf - 2 * c_inf / g1)
    vnb = 0.5 * (Rp + Rm)
    cb = 0.25 * g1 * (Rp - Rm)
    inflow = vnb < 0
    s_b = np.where(inflow, p_inf / rho_inf ** gamma, p / rho ** gamma)
    vb = np.stack([np.where(inflow, v_inf[i] + (vnb - vn_inf) * n[i], v[i] + (vnb - vn) * n[i]) for i in range(3)])
    rho_b = (cb * cb / (gamma * s_b)) ** (1.0 / g1)
    p_b = rho_b * cb * cb / gamma
    E_b = p_b / g1 + 0.5 * rho_b * (vb[0] ** 2 + vb[1] ** 2 + vb[2] ** 2)
    return np.stack([rho_b, rho_b * vb[0], rho_b * vb[1], rho_b * vb[2], E_b])


# ----------------------------------------------------------------------------- gather / scatter
def _gather(arrs, et, fpt, ele):
    """arrs: per type [N_f, V, N_e] -> [V, n] at the listed (type, flux point, element)."""
    out = np.empty((arrs[0].shape[1], len(et)))
    for t, a in enumerate(arrs):
        m = et == t
        if m.any():
            out[:, m] = a[fpt[m], :, ele[m]].T
    return out


def _scatter(arrs, et, fpt, ele, vals):
    for t, a in enumerate(arrs):
        m = et == t
        if m.any():
            a[fpt[m], :, ele[m]] = vals[:, m].T


def _apply(A, B):
    """Operator application C <- A B on a state matrix (eq. 1 with c1=1, c2=0):
    A [M, K], B [K, V, N_e] viewed as the row-major K x (V N_e) matrix."""
    K = B.shape[0]
    return (A @ B.reshape(K, -1)).reshape((A.shape[0],) + B.shape[1:])


# ----------------------------------------------------------------------------- right-hand side
def rhs(cfg, eles, ifc, bcs, us, parts=None, halo=None):
    """One evaluation of d u / d t, steps 1-6 of SURVEY 8(c).  If `parts` is a dict it receives the
    intermediates `ftil` (F~) and `d` (D) of step 6, for a-priori round-off bounds in the tests.

    halo (domain decomposition: "exchange of interface data between ranks"): dict(et, fpt, ele,
    exchange).  The flux-point pairs cut by the partition refer to their remote side as flux point 0 of element g of an extra
    pseudo type with index len(eles); halo['exchange'](name, values [V, n_send]) -> [V, n_ghost] hands the own values at the
    flux points (et, fpt, ele) to the peers and returns theirs -- once for U_f after step 1 and, for Navier-Stokes, once for the
    three components of G_f after step 3.  No arithmetic is added: the ghost values enter steps 2 and 5 as any other side.

    cfg  : dict(system='euler'|'ns', gamma, mu, prandtl, ldg_beta, ldg_tau)
    eles : per element type dict(M0, M132, M3, M460, M6, smats [3,3,N_u,N_e], rcpdjac [N_u,N_e])
    ifc  : dict(l_et,l_fpt,l_ele,r_et,r_fpt,r_ele, nl [3,n], magl [n], magr [n])
    bcs  : list of dict(type='wall'|'farfield', et,fpt,ele, n [3,nb], mag [nb], params)
    us   : per element type U [N_u, 5, N_e]
    """
    ns = cfg["system"] == "ns"
    gamma = cfg["gamma"]
    beta, tau = (cfg["ldg_beta"], cfg["ldg_tau"]) if ns else (0.0, 0.0)
    mu, pr = cfg.get("mu", 0.0), cfg.get("prandtl", 0.72)
    L = (ifc["l_et"], ifc["l_fpt"], ifc["l_ele"])
    R = (ifc["r_et"], ifc["r_fpt"], ifc["r_ele"])

    # step 1: U_f = M0 U
    uf = [_apply(e["M0"], u) for e, u in zip(eles, us)]
    if halo is not None:
        H = (halo["et"], halo["fpt"], halo["ele"])
        uf.append(halo["exchange"]("u", _gather(uf, *H))[None])          # ghost "type": [1 flux point, 5, n_ghost]
    uL, uR = _gather(uf, *L), _gather(uf, *R)

    def bc_states(b):
        ubL = _gather(uf, b["et"], b["fpt"], b["ele"])
        if b["type"] == "wall":
            ub, uv = ghost_wall(ubL, b["params"][0])
        elif b["type"] == "farfield":
            pr_ = b["params"]
            ub = ghost_farfield(ubL, b["n"], gamma, pr_[0], np.array(pr_[1:4]), pr_[4])
            uv = ub
        else:
            raise ValueError(b["type"])
        return ubL, ub, uv

    gf = None
    if ns:
        # step 2: common solution C = (1/2-beta) u_L + (1/2+beta) u_R at both sides; boundaries C = u_b^visc
        cf = [np.zeros_like(a) for a in uf]
        C = (0.5 - beta) * uL + (0.5 + beta) * uR
        _scatter(cf, *L, C)
        _scatter(cf, *R, C)
        for b in bcs:
            _, _, uv = bc_states(b)
            _scatter(cf, b["et"], b["fpt"], b["ele"], uv)
        # step 3: G~ = M460 U + M6 C ; G_i = (1/|J|) sum_alpha S[alpha,i] G~_alpha ; G_f,i = M0 G_i
        grads, gf = [], []
        for e, u, c in zip(eles, us, cf):
            nu = u.shape[0]
            gt = (_apply(e["M460"], u) + _apply(e["M6"], c)).reshape((3, nu) + u.shape[1:])
            S, rj = e["smats"], e["rcpdjac"]
            g = np.stack([rj[:, None, :] * sum(S[a, i][:, None, :] * gt[a] for a in range(3)) for i in range(3)])
            grads.append(g)
            gf.append(np.stack([_apply(e["M0"], g[i]) for i in range(3)]))
        if halo is not None:
            own = np.concatenate([_gather([g[i] for g in gf], *H) for i in range(3)])          # [15, n_send]
            gf.append(halo["exchange"]("g", own).reshape(3, 1, 5, -1))

    # step 4: transformed flux F~_alpha = sum_i S[alpha,i] (f^inv_i - f^visc_i)
    ftil = []
    for k, (e, u) in enumerate(zip(eles, us)):
        uu = u.transpose(1, 0, 2)                                      # [5, N_u, N_e]
        f = inviscid_flux(uu, gamma)
        if ns:
            f = f - viscous_flux(uu, grads[k].transpose(0, 2, 1, 3), gamma, mu, pr)
        S = e["smats"]
        ft = np.stack([sum(S[a, i][None] * f[i] for i in range(3)) for a in range(3)])    # [3, 5, N_u, N_e]
        ftil.append(ft.transpose(0, 2, 1, 3))                          # [3, N_u, 5, N_e]

    # step 5: common normal flux at interior pairs and boundary flux points
    d = [np.zeros_like(a) for a in uf]
    n = ifc["nl"]
    Fc = rusanov(uL, uR, n, gamma)
    if ns:
        qL = np.stack([_gather([g[i] for g in gf], *L) for i in range(3)])
        qR = np.stack([_gather([g[i] for g in gf], *R) for i in range(3)])
        fvL, fvR = viscous_flux(uL, qL, gamma, mu, pr), viscous_flux(uR, qR, gamma, mu, pr)
        Fc = Fc - sum(((0.5 + beta) * fvL[i] + (0.5 - beta) * fvR[i]) * n[i] for i in range(3)) + tau * (uL - uR)
    _scatter(d, *L, ifc["magl"] * Fc)
    _scatter(d, *R, -ifc["magr"] * Fc)
    for b in bcs:
        ubL, ub, uv = bc_states(b)
        Fb = rusanov(ubL, ub, b["n"], gamma)
        if ns:
            qb = np.stack([_gather([g[i] for g in gf], b["et"], b["fpt"], b["ele"]) for i in range(3)])
            fv = viscous_flux(uv, qb, gamma, mu, pr)
            Fb = Fb - sum(fv[i] * b["n"][i] for i in range(3)) + tau * (ubL - uv)
        _scatter(d, b["et"], b["fpt"], b["ele"], b["mag"] * Fb)

    if parts is not None:
        parts.update(ftil=ftil, d=d)
    # step 6: R = M132 F~ + M3 D ; dudt = -R / |J|
    out = []
    for e, ft, dd in zip(eles, ftil, d):
        nu = e["M132"].shape[0]
        r = _apply(e["M132"], ft.reshape((3 * nu,) + ft.shape[2:])) + _apply(e["M3"], dd)
        out.append(-r * e["rcpdjac"][:, None, :])
    return out


# ----------------------------------------------------------------------------- time steppers
def euler_step(f, us, dt):
    """Forward Euler (Table 1, "Time Steppers: Euler, RK4, RK45"): u <- u + dt f(u)."""
    return [u + dt * k for u, k in zip(us, f(us))]


def rk4_step(f, us, dt):
    """Classical RK4 (Table 1). `f(list of U) -> list of dU/dt`."""
    k1 = f(us)
    k2 = f([u + 0.5 * dt * k for u, k in zip(us, k1)])
    k3 = f([u + 0.5 * dt * k for u, k in zip(us, k2)])
    k4 = f([u + dt * k for u, k in zip(us, k3)])
    return [u + dt / 6.0 * (a + 2 * b + 2 * c + d) for u, a, b, c, d in zip(us, k1, k2, k3, k4)]


# RK4(3)5[2R+]C of Kennedy, Carpenter & Lewis (ref [23] PAPER.md:291); the
# coefficients are not printed in the paper (reading R12) and are pinned by the exact order
# conditions in tests/test_rk.py.
RK45_A = (970286171893 / 4311952581923, 6584761158862 / 12103376702013,
          2251764453980 / 15575788980749, 26877169314380 / 34165994151039)
RK45_B = (1153189308089 / 22510343858157, 1772645290293 / 4653164025191, -1672844663538 / 4480602732383,
          2114624349019 / 3568978502595, 5198255086312 / 14908931495163)
RK45_A_FRAC = ((970286171893, 4311952581923), (6584761158862, 12103376702013),
               (2251764453980, 15575788980749), (26877169314380, 34165994151039))
RK45_B_FRAC = ((1153189308089, 22510343858157), (1772645290293, 4653164025191), (-1672844663538, 4480602732383),
               (2114624349019, 3568978502595), (5198255086312, 14908931495163))


def rk45_step(f, us, dt):
    """RK45[2R+] in two-register van der Houwen form, fixed dt:
    X <- u; Y <- u; for i = 1..5: K <- f(Y); X <- X + dt b_i K; if i < 5: Y <- X + dt (a_i - b_i) K."""
    X = [u.copy() for u in us]
    Y = [u.copy() for u in us]
    for i in range(5):
        K = f(Y)
        X = [x + dt * RK45_B[i] * k for x, k in zip(X, K)]
        if i < 4:
            Y = [x + dt * (RK45_A[i] - RK45_B[i]) * k for x, k in zip(X, K)]
    return X


# Embedded third-order weights of RK4(3)5[2R+]C (PAPER.md:116 names the pair, not printed in the paper:
# reading R12); pinned by the exact order-3 conditions in tests/test_rk.py.
RK45_BHAT_FRAC = ((1016888040809, 7410784769900), (11231460423587, 58533540763752), (-1563879915014, 6823010717585),
                  (606302364029, 971179775848), (1097981568119, 3980877426909))
RK45_BHAT = tuple(n / d for n, d in RK45_BHAT_FRAC)


def rk45_step_with_error(f, us, dt):
    """One RK45[2R+] step and the embedded error estimate, from the definition: with the five stage derivatives K_i,
    u+ = u + dt sum b_i K_i,  E = dt sum (b_i - bhat_i) K_i  (difference between the fourth- and the third-order solution)."""
    X = [u.copy() for u in us]
    Y = [u.copy() for u in us]
    Ks = []
    for i in range(5):
        K = f(Y)
        Ks.append(K)
        X = [x + dt * RK45_B[i] * k for x, k in zip(X, K)]
        if i < 4:
            Y = [x + dt * (RK45_A[i] - RK45_B[i]) * k for x, k in zip(X, K)]
    E = [np.zeros_like(u) for u in us]
    for i in range(5):
        E = [e + dt * (RK45_B[i] - RK45_BHAT[i]) * k for e, k in zip(E, Ks[i])]
    return X, E


def error_norm(E, u_old, u_new, atol, rtol):
    """Reading R25: err = sqrt( mean over every solution point and variable of (E / (atol + rtol max(|u_n|, |u_n+1|)))^2 )."""
    s, n = 0.0, 0
    for e, a, b in zip(E, u_old, u_new):
        s += float(np.sum((np.abs(e) / (atol + rtol * np.maximum(np.abs(a), np.abs(b)))) ** 2))
        n += e.size
    return float(np.sqrt(s / n))


PI_ALPHA, PI_BETA, PI_SAFETY, PI_FMIN, PI_FMAX = 0.7 / 4, 0.4 / 4, 0.8, 0.3, 2.5


def pi_factor(err, err_prev):
    """Step-size factor of the PI controller (reading R25; Gustafsson's controller as in Hairer & Wanner II, IV.2, for a
    local error of order 4): clip(safety * err^-alpha * err_prev^beta, fmin, fmax); a non-finite error gives fmin."""
    if not np.isfinite(err):
        return PI_FMIN
    err = max(err, 1e-10)
    return float(min(PI_FMAX, max(PI_FMIN, PI_SAFETY * err ** (-PI_ALPHA) * err_prev ** PI_BETA)))


def rk45_adaptive(f, us, t0, t1, dt0, atol, rtol, max_attempts=10000):
    """Adaptive RK45[2R+] from t0 to t1 (reading R25).  Each attempt uses dt = min(dt, t1 - t); it is
    accepted iff err <= 1 (then t += dt, and t = t1 exactly when the step was cut to reach it); after every attempt
    dt <- dt * pi_factor(err, err_prev), err_prev being the error of the last accepted step (1 initially).
    Returns (state, history) with history = list of (dt tried, err, accepted)."""
    t, dt, err_prev = t0, dt0, 1.0
    hist = []
    us = [u.copy() for u in us]
    while t1 - t > 1e-12 * abs(t1 - t0) and len(hist) < max_attempts:
        last = dt >= t1 - t
        dtt = (t1 - t) if last else dt
        new, E = rk45_step_with_error(f, us, dtt)
        err = error_norm(E, us, new, atol, rtol)
        ok = bool(np.isfinite(err) and err <= 1.0)
        hist.append((dtt, err, ok))
        if ok:
            us = new
            t = t1 if last else t + dtt
        dt = dtt * pi_factor(err, err_prev)
        if ok:
            err_prev = max(err, 1e-10)
    return us, hist
