"""Reference elements, point sets and the constant FR operator matrices.

These are INPUTS of the hot path: `fr_setup(mesh, order, operator matrices, precision)`
(BASELINE.json north_star) takes the operators as dense FP64 host arrays, and the CPU oracle
takes the very same arrays.  The paper only names the volume-to-surface interpolation
operator M0 and gives its dimensions (Table 2); the remaining
operators follow the standard FR factorisation the paper defers to its refs [4], [8]
 -- written out in SURVEY.md Appendix A.4 and DESIGN.md "Readings" R4, R6, R7.

Construction: monomial basis on the unit (shifted) reference element, closed-form monomial
integrals (no quadrature), all O(N^3) linear algebra in double-double so that every entry is
a correctly rounded FP64 number.  Nothing here evaluates a flux or a right-hand side.

Conventions (all reference coordinates in [-1, 1]):
  tet   v0(-1,-1,-1) v1(1,-1,-1) v2(-1,1,-1) v3(-1,-1,1); faces (v0v1v2)(v0v1v3)(v0v2v3)(v1v2v3)
  pri   triangle (-1,-1),(1,-1),(-1,1) in (r,s) x t in [-1,1]; faces bottom, top, s=-1, r+s=0, r=-1
  hex   [-1,1]^3; faces t=-1, t=1, s=-1, r=1, s=1, r=-1
  row / column blocks of the stacked operators are alpha-major: (alpha, rho) -> alpha*N_u + rho
"""
from functools import lru_cache

import mpmath as mp
import numpy as np

from .ddmath import DD, dd_inv, dd_matmul, dd_pow

_DPS = 50

# ----------------------------------------------------------------------------- element topology
_VERTS = {
    "tet": [(-1, -1, -1), (1, -1, -1), (-1, 1, -1), (-1, -1, 1)],
    "pri": [(-1, -1, -1), (1, -1, -1), (-1, 1, -1), (-1, -1, 1), (1, -1, 1), (-1, 1, 1)],
    "hex": [(-1, -1, -1), (1, -1, -1), (1, 1, -1), (-1, 1, -1), (-1, -1, 1), (1, -1, 1), (1, 1, 1), (-1, 1, 1)],
}
# faces as local vertex tuples; 3 vertices = triangle (A,B,C), 4 = quad in cyclic order (A,B,C,D)
_FACES = {
    "tet": [(0, 1, 2), (0, 1, 3), (0, 2, 3), (1, 2, 3)],
    "pri": [(0, 1, 2), (3, 4, 5), (0, 1, 4, 3), (1, 2, 5, 4), (0, 2, 5, 3)],
    "hex": [(0, 1, 2, 3), (4, 5, 6, 7), (0, 1, 5, 4), (1, 2, 6, 5), (3, 2, 6, 7), (0, 3, 7, 4)],
}


def verts(etype):
    return np.array(_VERTS[etype], dtype=np.float64)


def faces(etype):
    return list(_FACES[etype])


def npts(etype, p):
    """(N_u, N_f) -- Table 2 of the paper."""
    t = (p + 1) * (p + 2) // 2
    q = (p + 1) ** 2
    if etype == "tet":
        return (p + 1) * (p + 2) * (p + 3) // 6, 4 * t
    if etype == "pri":
        return t * (p + 1), 2 * t + 3 * q
    if etype == "hex":
        return (p + 1) ** 3, 6 * q
    raise ValueError(etype)


# ----------------------------------------------------------------------------- point sets (mp)
def _gl_mp(n):
    """n Gauss-Legendre nodes on (-1,1), ascending, as mpmath numbers (Newton on P_n)."""
    x0 = np.sort(np.polynomial.legendre.leggauss(n)[0])
    out = []
    for x in x0:
        x = mp.mpf(float(x))
        for _ in range(8):
            p0, p1 = mp.mpf(1), x
            for k in range(2, n + 1):
                p0, p1 = p1, ((2 * k - 1) * x * p1 - (k - 1) * p0) / k
            dp = n * (x * p1 - p0) / (x * x - 1)
            x = x - p1 / dp
        out.append(x)
    return out


def _tri_pts_mp(p):
    """Blyth-Pozrikidis-type symmetric triangle set on the GL nodes (reading R6)."""
    g = _gl_mp(p + 1)
    v = [(1 + x) / 2 for x in g]
    pts = []
    for i in range(p + 1):
        for j in range(p + 1 - i):
            k = p - i - j
            idx = (i, j, k)
            lam = [(1 + 2 * v[idx[a]] - sum(v[idx[b]] for b in range(3) if b != a)) / 3 for a in range(3)]
            pts.append((2 * lam[1] - 1, 2 * lam[2] - 1))
    return pts


def _tet_pts_mp(p):
    g = _gl_mp(p + 1)
    v = [(1 + x) / 2 for x in g]
    pts = []
    for i in range(p + 1):
        for j in range(p + 1 - i):
            for k in range(p + 1 - i - j):
                l = p - i - j - k
                idx = (i, j, k, l)
                lam = [(1 + 3 * v[idx[a]] - sum(v[idx[b]] for b in range(4) if b != a)) / 4 for a in range(4)]
                pts.append((2 * lam[1] - 1, 2 * lam[2] - 1, 2 * lam[3] - 1))
    return pts


def _quad_pts_mp(p):
    g = _gl_mp(p + 1)
    return [(g[i], g[j]) for j in range(p + 1) for i in range(p + 1)]


def _upts_mp(etype, p):
    g = _gl_mp(p + 1)
    if etype == "tet":
        return _tet_pts_mp(p)
    if etype == "pri":
        tri = _tri_pts_mp(p)
        return [(r, s, g[b]) for b in range(p + 1) for (r, s) in tri]
    if etype == "hex":
        return [(g[i], g[j], g[k]) for k in range(p + 1) for j in range(p + 1) for i in range(p + 1)]
    raise ValueError(etype)


def _face_geometry_mp(etype):
    """Per face: (vertex tuple, unit outward reference normal, area factor a_f)."""
    V = [tuple(mp.mpf(c) for c in v) for v in _VERTS[etype]]
    cen = [sum(v[d] for v in V) / len(V) for d in range(3)]
    out = []
    for fv in _FACES[etype]:
        A, B = V[fv[0]], V[fv[1]]
        Dv = V[fv[-1]]  # C for a triangle, D for a quad: the second edge from A
        e1 = [B[d] - A[d] for d in range(3)]
        e2 = [Dv[d] - A[d] for d in range(3)]
        cr = [e1[1] * e2[2] - e1[2] * e2[1], e1[2] * e2[0] - e1[0] * e2[2], e1[0] * e2[1] - e1[1] * e2[0]]
        nrm = mp.sqrt(sum(c * c for c in cr))
        n = [c / nrm for c in cr]
        fc = [sum(V[i][d] for i in fv) / len(fv) for d in range(3)]
        if sum(n[d] * (fc[d] - cen[d]) for d in range(3)) < 0:
            n = [-c for c in n]
        # triangle: area = |cr|/2, reference triangle area 2; quad (parallelogram): |cr|, reference 4
        a_f = nrm / 4
        out.append((fv, n, a_f))
    return out


def _place_on_face(V, fv, ab):
    a, b = ab
    if len(fv) == 3:
        A, B, C = (V[i] for i in fv)
        return tuple(A[d] + (a + 1) / 2 * (B[d] - A[d]) + (b + 1) / 2 * (C[d] - A[d]) for d in range(3))
    A, B, C, Dv = (V[i] for i in fv)
    return tuple(((1 - a) * (1 - b) * A[d] + (1 + a) * (1 - b) * B[d] + (1 + a) * (1 + b) * C[d]
                  + (1 - a) * (1 + b) * Dv[d]) / 4 for d in range(3))


# ----------------------------------------------------------------------------- monomial spaces
def _exps3(etype, p):
    if etype == "tet":
        return [(a, b, c) for a in range(p + 1) for b in range(p + 1 - a) for c in range(p + 1 - a - b)]
    if etype == "pri":
        return [(a, b, c) for a in range(p + 1) for b in range(p + 1 - a) for c in range(p + 1)]
    return [(a, b, c) for a in range(p + 1) for b in range(p + 1) for c in range(p + 1)]


def _exps2(tri, p):
    if tri:
        return [(a, b) for a in range(p + 1) for b in range(p + 1 - a)]
    return [(a, b) for a in range(p + 1) for b in range(p + 1)]


def _int3(etype, e):
    """Integral of x^a y^b z^c over the unit (shifted) reference element, exact (mp)."""
    a, b, c = e
    f = mp.factorial
    if etype == "tet":
        return f(a) * f(b) * f(c) / f(a + b + c + 3)
    if etype == "pri":
        return f(a) * f(b) / f(a + b + 2) / (c + 1)
    return mp.mpf(1) / ((a + 1) * (b + 1) * (c + 1))


def _int2(tri, e):
    a, b = e
    f = mp.factorial
    if tri:
        return f(a) * f(b) / f(a + b + 2)
    return mp.mpf(1) / ((a + 1) * (b + 1))


def _vander(pts_dd, exps, deriv=None):
    """Monomials prod_d x_d^e_d at shifted points x=(r+1)/2; optional d/dr_deriv (factor 1/2 included)."""
    n = pts_dd.shape[0]
    out = None
    E = np.array(exps, dtype=np.int64)
    coef = np.ones(len(exps))
    E = E.copy()
    if deriv is not None:
        coef = 0.5 * E[:, deriv].astype(np.float64)
        E[:, deriv] = np.maximum(E[:, deriv] - 1, 0)
    for d in range(E.shape[1]):
        x = DD(np.repeat(pts_dd.hi[:, d:d + 1], len(exps), axis=1), np.repeat(pts_dd.lo[:, d:d + 1], len(exps), axis=1))
        term = dd_pow(x, np.broadcast_to(E[None, :, d], (n, len(exps))))
        out = term if out is None else out * term
    return out * DD(np.broadcast_to(coef[None, :], (n, len(exps))).copy())


def _shift(pts_mp):
    return DD.from_mp([[(c + 1) / 2 for c in pt] for pt in pts_mp])


# ----------------------------------------------------------------------------- operators
@lru_cache(maxsize=None)
def operators(etype, p):
    """All constant per-(element type, order) data, FP64 numpy arrays in a dict.

    upts [N_u,3], fpts [N_f,3], fnorm [N_f,3] unit reference normals, fface [N_f] face of each
    flux point, faces (vertex tuples), face_area_factor, wts [N_u] (omega = int l_rho),
    fwts [N_f] (w_sigma = a_f int_face l^face_sigma), and
    M0 [N_f,N_u]  M1 [N_u,3N_u]  M2 [N_f,3N_u]  M3 [N_u,N_f]  M4 [3N_u,N_u]  M6 [3N_u,N_f]
    M132 = M1 - M3 M2,  M460 = M4 - M6 M0   (the "applied" operators).
    """
    if etype not in _VERTS:
        raise ValueError(etype)
    if p < 1:
        raise ValueError("order must be >= 1")
    with mp.workdps(_DPS):
        nu, nf = npts(etype, p)
        up = _upts_mp(etype, p)
        assert len(up) == nu
        Vm = [tuple(mp.mpf(c) for c in v) for v in _VERTS[etype]]
        fgeo = _face_geometry_mp(etype)
        fp, fn, fface, fab = [], [], [], []
        face_sets = []
        for fi, (fv, n, a_f) in enumerate(fgeo):
            pts2 = _tri_pts_mp(p) if len(fv) == 3 else _quad_pts_mp(p)
            face_sets.append(pts2)
            for ab in pts2:
                fp.append(_place_on_face(Vm, fv, ab))
                fn.append(n)
                fface.append(fi)
                fab.append(ab)
        assert len(fp) == nf
        ex3 = _exps3(etype, p)
        assert len(ex3) == nu
        g3 = DD.from_mp([_int3(etype, e) for e in ex3])
        G3 = DD.from_mp([[_int3(etype, tuple(x + y for x, y in zip(e1, e2))) for e2 in ex3] for e1 in ex3])
        up_dd, fp_dd = _shift(up), _shift(fp)
        fn_dd = DD.from_mp(fn)
        face_data = []
        for fi, (fv, n, a_f) in enumerate(fgeo):
            tri = len(fv) == 3
            ex2 = _exps2(tri, p)
            g2 = DD.from_mp([_int2(tri, e) for e in ex2])
            G2 = DD.from_mp([[_int2(tri, (e1[0] + e2[0], e1[1] + e2[1])) for e2 in ex2] for e1 in ex2])
            face_data.append((ex2, g2, G2, DD.from_mp([a_f]), _shift(face_sets[fi])))

    V = _vander(up_dd, ex3)
    Vinv = dd_inv(V)
    M0 = dd_matmul(_vander(fp_dd, ex3), Vinv)
    M4b = [dd_matmul(_vander(up_dd, ex3, deriv=a), Vinv) for a in range(3)]
    # Mass = Vinv^T (8 G) Vinv  =>  Mass^-1 = V (8 G)^-1 V^T
    Ginv = dd_inv(G3)
    Minv = dd_matmul(dd_matmul(V, Ginv), V.T) * DD(np.full((nu, nu), 0.125))
    wts = dd_matmul(Vinv.T, g3.reshape(nu, 1)) * DD(np.full((nu, 1), 8.0))

    B = DD(np.zeros((nu, nf)))
    fwts = DD(np.zeros(nf))
    fface = np.array(fface)
    for fi, (ex2, g2, G2, a_f, pts2) in enumerate(face_data):
        sel = np.nonzero(fface == fi)[0]
        nfp = len(sel)
        V2inv = dd_inv(_vander(pts2, ex2))
        four_af = a_f * DD(np.array([4.0]))
        Mf = dd_matmul(dd_matmul(V2inv.T, G2), V2inv) * DD(np.broadcast_to(four_af.hi, (nfp, nfp)).copy(),
                                                             np.broadcast_to(four_af.lo, (nfp, nfp)).copy())
        Bf = dd_matmul(M0[sel].T, Mf)
        B.hi[:, sel] = Bf.hi
        B.lo[:, sel] = Bf.lo
        wf = dd_matmul(V2inv.T, g2.reshape(nfp, 1)) * DD(np.broadcast_to(four_af.hi, (nfp, 1)).copy(),
                                                         np.broadcast_to(four_af.lo, (nfp, 1)).copy())
        fwts.hi[sel] = wf.hi[:, 0]
        fwts.lo[sel] = wf.lo[:, 0]
    M3 = dd_matmul(Minv, B)

    def _hstack(blocks):
        return DD(np.concatenate([b.hi for b in blocks], axis=1), np.concatenate([b.lo for b in blocks], axis=1))

    def _vstack(blocks):
        return DD(np.concatenate([b.hi for b in blocks], axis=0), np.concatenate([b.lo for b in blocks], axis=0))

    def _rowscale(mat, col):  # mat[sigma, :] * col[sigma]
        return mat * DD(np.repeat(col.hi[:, None], mat.shape[1], axis=1), np.repeat(col.lo[:, None], mat.shape[1], axis=1))

    def _colscale(mat, row):  # mat[:, sigma] * row[sigma]
        return mat * DD(np.repeat(row.hi[None, :], mat.shape[0], axis=0), np.repeat(row.lo[None, :], mat.shape[0], axis=0))

    M4 = _vstack(M4b)
    M1 = _hstack(M4b)
    M2 = _hstack([_rowscale(M0, fn_dd[:, a]) for a in range(3)])
    M6 = _vstack([_colscale(M3, fn_dd[:, a]) for a in range(3)])
    M132 = M1 - dd_matmul(M3, M2)
    M460 = M4 - dd_matmul(M6, M0)

    f64 = lambda x: np.ascontiguousarray(x.to_f64())
    out = dict(
        etype=etype, order=p, nupts=nu, nfpts=nf,
        upts=np.array([[float(c) for c in pt] for pt in up]),
        fpts=np.array([[float(c) for c in pt] for pt in fp]),
        fab=np.array([[float(c) for c in ab] for ab in fab]),
        fnorm=f64(fn_dd), fface=fface.astype(np.int32),
        faces=faces(etype), face_area_factor=np.array([float(a.to_f64()[0]) for (_, _, _, a, _) in face_data]),
        wts=f64(wts)[:, 0], fwts=f64(fwts),
        M0=f64(M0), M1=f64(M1), M2=f64(M2), M3=f64(M3), M4=f64(M4), M6=f64(M6), M132=f64(M132), M460=f64(M460),
    )
    for v in out.values():
        if isinstance(v, np.ndarray):
            v.setflags(write=False)
    return out
