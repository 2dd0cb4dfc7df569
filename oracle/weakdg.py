"""CPU ORACLE, second formulation -- TEST INFRASTRUCTURE, NOT PRODUCT CODE.

Brute-force weak nodal-DG evaluation of the same right-hand side, used to pin `oracle.fr_oracle.rhs`
(and, through it, the operator matrices handed to `fr_setup`) on few-element meshes (BASELINE.json
north_star: "brute-force agreement on a few-element mesh").

The paper states that FR "incorporates ... the nodal DG schemes" and that a DG scheme was
used.  FR with DG correction functions must therefore reproduce, to round-off,

    |J| Mass dU/dt = sum_alpha K_alpha F~_alpha - B D ,         Mass G~_alpha = -K_alpha U + B_alpha C ,

with Mass[r,n] = int l_r l_n, K_alpha[r,n] = int d_alpha(l_r) l_n, B[r,s] = int_face l_r l^face_s and
B_alpha = B n^_alpha -- no M1/M2/M3/M4/M6 anywhere.  Everything here is built independently of
`fr_inputs.refelem`'s operator code: own nodal basis (monomial Vandermonde in FP64), own Gauss-Jacobi
quadrature, own face normals / area factors, and own *scalar* (one point at a time, pure Python)
physics: ideal-gas Euler flux, Newtonian viscous flux written from PRIMITIVE-variable gradients,
Rusanov flux, LDG common values.  Only the point sets and the element topology (conventions) are
taken as inputs.  Small meshes and p <= 3 only (monomial conditioning, Python loops).
"""
import math

import numpy as np
from scipy.special import roots_jacobi

# ----------------------------------------------------------------------------- quadrature


def _gj01(n, alpha):
    """Gauss-Jacobi nodes/weights on [0,1] for the weight (1-u)^alpha."""
    x, w = roots_jacobi(n, alpha, 0)
    return (x + 1) / 2, w / 2 ** (alpha + 1)


def quad_tri(n):
    """Reference triangle (-1,-1),(1,-1),(-1,1): points [m,2], weights (sum = 2)."""
    u, wu = _gj01(n, 1)
    v, wv = _gj01(n, 0)
    pts, wts = [], []
    for a, wa in zip(u, wu):
        for b, wb in zip(v, wv):
            x, y = a, b * (1 - a)
            pts.append((2 * x - 1, 2 * y - 1))
            wts.append(4 * wa * wb)
    return np.array(pts), np.array(wts)


def quad_line(n):
    x, w = roots_jacobi(n, 0, 0)
    return x, w


def quad_volume(etype, n):
    if etype == "tet":
        u, wu = _gj01(n, 2)
        v, wv = _gj01(n, 1)
        w_, ww = _gj01(n, 0)
        pts, wts = [], []
        for a, wa in zip(u, wu):
            for b, wb in zip(v, wv):
                for c, wc in zip(w_, ww):
                    x, y, z = a, b * (1 - a), c * (1 - a) * (1 - b)
                    pts.append((2 * x - 1, 2 * y - 1, 2 * z - 1))
                    wts.append(8 * wa * wb * wc)
        return np.array(pts), np.array(wts)
    if etype == "pri":
        tp, tw = quad_tri(n)
        lx, lw = quad_line(n)
        pts = [(r, s, t) for (r, s) in tp for t in lx]
        wts = [a * b for a in tw for b in lw]
        return np.array(pts), np.array(wts)
    raise ValueError(etype)


# ----------------------------------------------------------------------------- own nodal bases
def _exps(etype, p):
    if etype == "tet":
        return [(a, b, c) for a in range(p + 1) for b in range(p + 1) for c in range(p + 1) if a + b + c <= p]
    if etype == "pri":
        return [(a, b, c) for a in range(p + 1) for b in range(p + 1) for c in range(p + 1) if a + b <= p]
    if etype == "tri":
        return [(a, b) for a in range(p + 1) for b in range(p + 1) if a + b <= p]
    if etype == "quad":
        return [(a, b) for a in range(p + 1) for b in range(p + 1)]
    raise ValueError(etype)


def _vand(x, ex, d=None):
    x = np.atleast_2d(x)
    cols = []
    for e in ex:
        c = np.ones(x.shape[0])
        for k, ek in enumerate(e):
            if d == k:
                c = c * (ek * x[:, k] ** (ek - 1) if ek > 0 else 0.0)
            else:
                c = c * x[:, k] ** ek
        cols.append(c)
    return np.stack(cols, axis=1)


class RefElement:
    """Mass, K_alpha, B, interpolation to flux points -- by quadrature with an own monomial nodal basis."""

    def __init__(self, etype, p, upts, fpts, fface, fab, verts, faces):
        self.etype, self.p = etype, p
        nu, nf = len(upts), len(fpts)
        ex = _exps(etype, p)
        assert len(ex) == nu
        Vi = np.linalg.inv(_vand(upts, ex))
        basis = lambda x: _vand(x, ex) @ Vi                        # [npts, N_u]
        dbasis = lambda x, a: _vand(x, ex, d=a) @ Vi
        qx, qw = quad_volume(etype, p + 2)
        L = basis(qx)
        self.mass = L.T @ (qw[:, None] * L)
        self.K = [dbasis(qx, a).T @ (qw[:, None] * L) for a in range(3)]
        self.interp = basis(fpts)                                   # [N_f, N_u]
        self.B = np.zeros((nu, nf))
        self.nhat = np.zeros((nf, 3))
        cen = verts.mean(axis=0)
        for fi, fv in enumerate(faces):
            sel = np.nonzero(fface == fi)[0]
            tri = len(fv) == 3
            ex2 = _exps("tri" if tri else "quad", p)
            V2i = np.linalg.inv(_vand(fab[sel], ex2))
            if tri:
                q2, w2 = quad_tri(p + 2)
                A, Bv, C = verts[list(fv)]
                place = lambda ab: A + np.outer((ab[:, 0] + 1) / 2, Bv - A) + np.outer((ab[:, 1] + 1) / 2, C - A)
                nrm = np.cross(Bv - A, C - A)
                area_factor = np.linalg.norm(nrm) / 2 / 2.0
            else:
                gx, gw = quad_line(p + 2)
                q2 = np.array([(a, b) for a in gx for b in gx])
                w2 = np.array([wa * wb for wa in gw for wb in gw])
                A, Bv, C, D = verts[list(fv)]
                place = lambda ab: ((1 - ab[:, :1]) * (1 - ab[:, 1:]) * A + (1 + ab[:, :1]) * (1 - ab[:, 1:]) * Bv
                                    + (1 + ab[:, :1]) * (1 + ab[:, 1:]) * C + (1 - ab[:, :1]) * (1 + ab[:, 1:]) * D) / 4
                nrm = np.cross(Bv - A, D - A)
                area_factor = np.linalg.norm(nrm) / 4.0
            nrm = nrm / np.linalg.norm(nrm)
            if nrm @ (verts[list(fv)].mean(axis=0) - cen) < 0:
                nrm = -nrm
            self.nhat[sel] = nrm
            Lvol = basis(place(q2))                                 # volume basis on the face quad points
            Lface = _vand(q2, ex2) @ V2i                            # face nodal basis
            self.B[:, sel] = area_factor * Lvol.T @ (w2[:, None] * Lface)


# ----------------------------------------------------------------------------- scalar physics
def _prim(u, gamma):
    rho = u[0]
    v = [u[1] / rho, u[2] / rho, u[3] / rho]
    p = (gamma - 1) * (u[4] - 0.5 * rho * (v[0] ** 2 + v[1] ** 2 + v[2] ** 2))
    return rho, v, p


def euler_flux_pt(u, gamma):
    rho, v, p = _prim(u, gamma)
    return [[rho * v[i], rho * v[i] * v[0] + (p if i == 0 else 0), rho * v[i] * v[1] + (p if i == 1 else 0),
             rho * v[i] * v[2] + (p if i == 2 else 0), (u[4] + p) * v[i]] for i in range(3)]


def viscous_flux_pt(u, q, gamma, mu, pr):
    """Textbook form from primitive gradients: tau_ij = mu (d_i v_j + d_j v_i - 2/3 delta_ij div v),
    heat flux kappa dT with kappa = mu c_p / Pr, T = p / (rho R); returned as f_i (5 components)."""
    rho, v, p = _prim(u, gamma)
    drho = [q[i][0] for i in range(3)]
    dv = [[(q[i][1 + j] - v[j] * drho[i]) / rho for j in range(3)] for i in range(3)]       # dv[i][j] = d_i v_j
    # p = (g-1)(E - m.m/(2 rho))  ->  d_i p
    dp = [(gamma - 1) * (q[i][4] - sum(v[j] * q[i][1 + j] for j in range(3)) + 0.5 * sum(c * c for c in v) * drho[i])
          for i in range(3)]
    # T = p / rho (R = 1), c_p = gamma/(gamma-1)
    dT = [(dp[i] - (p / rho) * drho[i]) / rho for i in range(3)]
    kappa = mu * gamma / (gamma - 1) / pr
    div = dv[0][0] + dv[1][1] + dv[2][2]
    out = []
    for i in range(3):
        tau = [mu * (dv[i][j] + dv[j][i] - (2.0 / 3.0) * div * (1 if i == j else 0)) for j in range(3)]
        out.append([0.0, tau[0], tau[1], tau[2], sum(v[j] * tau[j] for j in range(3)) + kappa * dT[i]])
    return out


def rusanov_pt(uL, uR, n, gamma):
    fL, fR = euler_flux_pt(uL, gamma), euler_flux_pt(uR, gamma)
    lam = 0.0
    for u in (uL, uR):
        rho, v, p = _prim(u, gamma)
        lam = max(lam, abs(sum(v[i] * n[i] for i in range(3))) + math.sqrt(gamma * p / rho))
    return [0.5 * sum((fL[i][k] + fR[i][k]) * n[i] for i in range(3)) + 0.5 * lam * (uL[k] - uR[k]) for k in range(5)]


# ----------------------------------------------------------------------------- brute-force RHS
def rhs(cfg, refs, eles, ifc, us):
    """Weak-DG right-hand side on a fully periodic mesh (no boundary conditions).

    refs : per type RefElement;  eles: per type dict(smats [3,3,N_u,N_e], rcpdjac [N_u,N_e]);
    ifc  : flux-point pairs with nl, magl, magr;  us: per type [N_u,5,N_e].
    """
    ns = cfg["system"] == "ns"
    gamma = cfg["gamma"]
    beta, tau = (cfg["ldg_beta"], cfg["ldg_tau"]) if ns else (0.0, 0.0)
    mu, pr = cfg.get("mu", 0.0), cfg.get("prandtl", 0.72)
    nt = len(us)
    npairs = len(ifc["l_et"])
    uf = [np.einsum("fu,uve->fve", r.interp, u) for r, u in zip(refs, us)]
    side = lambda arrs, s, k: arrs[ifc[s + "_et"][k]][ifc[s + "_fpt"][k], :, ifc[s + "_ele"][k]]

    grads = gf = None
    if ns:
        cf = [np.zeros_like(a) for a in uf]
        for k in range(npairs):
            uL, uR = side(uf, "l", k), side(uf, "r", k)
            c = (0.5 - beta) * uL + (0.5 + beta) * uR
            cf[ifc["l_et"][k]][ifc["l_fpt"][k], :, ifc["l_ele"][k]] = c
            cf[ifc["r_et"][k]][ifc["r_fpt"][k], :, ifc["r_ele"][k]] = c
        grads, gf = [], []
        for r, e, u, c in zip(refs, eles, us, cf):
            minv = np.linalg.inv(r.mass)
            gt = [np.einsum("mr,rve->mve", minv, -np.einsum("rn,nve->rve", r.K[a], u)
                            + np.einsum("rs,sve->rve", r.B * r.nhat[None, :, a], c)) for a in range(3)]
            S, rj = e["smats"], e["rcpdjac"]
            g = [rj[:, None, :] * sum(S[a, i][:, None, :] * gt[a] for a in range(3)) for i in range(3)]
            grads.append(g)
            gf.append([np.einsum("fu,uve->fve", r.interp, g[i]) for i in range(3)])

    ftil = []
    for t in range(nt):
        u, S = us[t], eles[t]["smats"]
        nu, _, ne = u.shape
        ft = np.zeros((3, nu, 5, ne))
        for rr in range(nu):
            for ee in range(ne):
                f = euler_flux_pt(u[rr, :, ee], gamma)
                if ns:
                    fv = viscous_flux_pt(u[rr, :, ee], [grads[t][i][rr, :, ee] for i in range(3)], gamma, mu, pr)
                    f = [[f[i][k] - fv[i][k] for k in range(5)] for i in range(3)]
                for a in range(3):
                    for k in range(5):
                        ft[a, rr, k, ee] = sum(S[a, i, rr, ee] * f[i][k] for i in range(3))
        ftil.append(ft)

    d = [np.zeros_like(a) for a in uf]
    for k in range(npairs):
        uL, uR = side(uf, "l", k), side(uf, "r", k)
        n = ifc["nl"][:, k]
        F = rusanov_pt(uL, uR, n, gamma)
        if ns:
            qL = [side([g[i] for g in gf], "l", k) for i in range(3)]
            qR = [side([g[i] for g in gf], "r", k) for i in range(3)]
            fvL, fvR = viscous_flux_pt(uL, qL, gamma, mu, pr), viscous_flux_pt(uR, qR, gamma, mu, pr)
            F = [F[m] - sum(((0.5 + beta) * fvL[i][m] + (0.5 - beta) * fvR[i][m]) * n[i] for i in range(3))
                 + tau * (uL[m] - uR[m]) for m in range(5)]
        F = np.array(F)
        d[ifc["l_et"][k]][ifc["l_fpt"][k], :, ifc["l_ele"][k]] = ifc["magl"][k] * F
        d[ifc["r_et"][k]][ifc["r_fpt"][k], :, ifc["r_ele"][k]] = -ifc["magr"][k] * F

    out = []
    for r, e, ft, dd in zip(refs, eles, ftil, d):
        rhs_ = sum(np.einsum("rn,nve->rve", r.K[a], ft[a]) for a in range(3)) - np.einsum("rs,sve->rve", r.B, dd)
        out.append(np.einsum("rn,nve->rve", np.linalg.inv(r.mass), rhs_) * e["rcpdjac"][:, None, :])
    return out
