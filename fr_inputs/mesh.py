"""Seeded synthetic mesh generators, element geometry and flux-point connectivity.

Inputs of the hot path only (the `mesh` argument of `fr_setup`, BASELINE.json north_star):
vertex coordinates -> metric terms (`smats`, `rcpdjac`), flux-point pairs, unit normals and
per-side magnitudes.  No flux, no operator application, no time stepping.

The paper's own meshes are not available; the generators follow the shapes
BASELINE.json configs[0..2] describe (recipe in DESIGN.md "Input recipe").

A mesh is a dict:
  etypes : list of element-type names; position = index into `eles[]` of the C ABI
  xv     : {etype: [N_e, n_vert, 3] float64 vertex coordinates (unwrapped across periodic seams)}
  xq     : optional {etype: [N_e, n_quad, 3]} quadratic node coordinates (`quad_nodes` order; the first n_vert are xv)
  vid    : {etype: [N_e, n_vert] int64 global vertex ids, identical across periodic images}
  period : length-3 list, period length per direction or None
  bc_tag : callable(face centroid [n,3]) -> int tag array, or None if the mesh is fully periodic
"""
import itertools

import numpy as np

from . import refelem

# ----------------------------------------------------------------------------- shape functions


def shape(etype, x):
    """Linear vertex shape functions N [npts, nv] and reference gradients dN [npts, nv, 3]."""
    x = np.asarray(x, dtype=np.float64)
    r, s, t = x[:, 0], x[:, 1], x[:, 2]
    o, z = np.ones_like(r), np.zeros_like(r)
    if etype == "tet":
        N = np.stack([-(1 + r + s + t) / 2, (1 + r) / 2, (1 + s) / 2, (1 + t) / 2], axis=1)
        dN = np.stack([np.stack([-o / 2, -o / 2, -o / 2], 1), np.stack([o / 2, z, z], 1),
                       np.stack([z, o / 2, z], 1), np.stack([z, z, o / 2], 1)], axis=1)
        return N, dN
    if etype == "pri":
        L = [-(r + s) / 2, (1 + r) / 2, (1 + s) / 2]
        dL = [(-o / 2, -o / 2), (o / 2, z), (z, o / 2)]
        lo, hi = (1 - t) / 2, (1 + t) / 2
        N = np.stack([L[0] * lo, L[1] * lo, L[2] * lo, L[0] * hi, L[1] * hi, L[2] * hi], axis=1)
        dN = np.stack([np.stack([dL[i][0] * lo, dL[i][1] * lo, -L[i] / 2], 1) for i in range(3)]
                      + [np.stack([dL[i][0] * hi, dL[i][1] * hi, L[i] / 2], 1) for i in range(3)], axis=1)
        return N, dN
    if etype == "hex":
        # trilinear, vertex order of refelem (bottom quad counter-clockwise, then top quad)
        sg = np.array(refelem._VERTS["hex"], dtype=np.float64)          # [8, 3] signs
        fr, fs, ft = (1 + sg[None, :, 0] * r[:, None]), (1 + sg[None, :, 1] * s[:, None]), (1 + sg[None, :, 2] * t[:, None])
        N = fr * fs * ft / 8
        dN = np.stack([sg[None, :, 0] * fs * ft, fr * sg[None, :, 1] * ft, fr * fs * sg[None, :, 2]], axis=2) / 8
        return N, dN
    raise ValueError(etype)


# quadratic (second-order, "quadratically curved") geometry: P2 tetrahedra (10 nodes), P2(tri) x P2(line) prisms
# (18 nodes), Q2 hexahedra (27 nodes).  Node order: the vertices first (order of `shape`), then the remaining nodes.
def _quad_exponents(etype):
    rng3 = range(3)
    if etype == "tet":
        return [(a, b, c) for a in rng3 for b in rng3 for c in rng3 if a + b + c <= 2]
    if etype == "pri":
        return [(a, b, c) for a in rng3 for b in rng3 for c in rng3 if a + b <= 2]
    if etype == "hex":
        return [(a, b, c) for a in rng3 for b in rng3 for c in rng3]
    raise ValueError(etype)


def quad_nodes(etype):
    """Reference coordinates [nq, 3] of the quadratic nodes: vertices, then edge midpoints (and, prism / hex, the face and
    cell centres that the tensor-product spaces carry)."""
    v = np.array(refelem._VERTS[etype], dtype=np.float64)
    if etype == "tet":
        rest = [(v[i] + v[j]) / 2 for i in range(4) for j in range(i + 1, 4)]
    elif etype == "pri":
        tri = v[:3, :2]
        t6 = [tri[0], tri[1], tri[2], (tri[0] + tri[1]) / 2, (tri[1] + tri[2]) / 2, (tri[0] + tri[2]) / 2]
        allp = [np.array([q[0], q[1], t]) for t in (-1.0, 1.0, 0.0) for q in t6]
        rest = [q for q in allp if not any(np.allclose(q, w) for w in v)]
    else:
        allp = [np.array([a, b, c]) for c in (-1.0, 0.0, 1.0) for b in (-1.0, 0.0, 1.0) for a in (-1.0, 0.0, 1.0)]
        rest = [q for q in allp if not any(np.allclose(q, w) for w in v)]
    return np.concatenate([v, np.array(rest)], axis=0)


def shape2(etype, x):
    """Quadratic nodal shape functions N [npts, nq] on `quad_nodes(etype)` and reference gradients dN [npts, nq, 3]."""
    x = np.asarray(x, dtype=np.float64)
    ex = _quad_exponents(etype)

    def mono(y):
        return np.stack([y[:, 0] ** a * y[:, 1] ** b * y[:, 2] ** c for a, b, c in ex], axis=1)

    def dmono(y):
        cols = []
        for a, b, c in ex:
            d0 = a * y[:, 0] ** max(a - 1, 0) * y[:, 1] ** b * y[:, 2] ** c if a else np.zeros(len(y))
            d1 = b * y[:, 0] ** a * y[:, 1] ** max(b - 1, 0) * y[:, 2] ** c if b else np.zeros(len(y))
            d2 = c * y[:, 0] ** a * y[:, 1] ** b * y[:, 2] ** max(c - 1, 0) if c else np.zeros(len(y))
            cols.append(np.stack([d0, d1, d2], axis=1))
        return np.stack(cols, axis=1)           # [npts, nmono, 3]

    Vinv = np.linalg.inv(mono(quad_nodes(etype)))
    return mono(x) @ Vinv, np.einsum("pma,mq->pqa", dmono(x), Vinv)


_NQUAD = {10: "tet", 18: "pri", 27: "hex"}


def curve_nodes(etype, xv, lat, fn, wfn=None):
    """Quadratic node coordinates [N_e, nq, 3] of elements that are straight in the parameter space `lat` ([N_e, nv, 3]) of a smooth
    map `fn`:  x_q = fn(lat_q) + sum_v N_v(q) (xv_v - fn(lat_v)),  lat_q = sum_v N_v(q) lat_v  (N = linear vertex shape functions).
    Vertices stay where they are; edge, face and cell nodes follow the map, so neighbours (which share the vertices, hence the
    parameter-space positions, of their common face) stay conforming.  `wfn(lat_q)` in [0, 1] optionally scales the departure
    from the straight element (1 = follow the map, 0 = stay straight), e.g. to curve only the elements near a wall."""
    N, _ = shape(etype, quad_nodes(etype))
    latq = np.einsum("qv,evi->eqi", N, lat)
    bend = fn(latq) - np.einsum("qv,evi->eqi", N, fn(lat))
    if wfn is not None:
        bend = bend * wfn(latq)[..., None]
    return np.einsum("qv,evi->eqi", N, xv) + bend


def _adjugate(J):
    """J [..., 3(i), 3(alpha)] -> S [..., 3(alpha), 3(i)] = det(J) * inv(J), and det(J)."""
    a, b, c = J[..., :, 0], J[..., :, 1], J[..., :, 2]
    S = np.stack([np.cross(b, c), np.cross(c, a), np.cross(a, b)], axis=-2)
    det = np.einsum("...i,...i->...", a, S[..., 0, :])
    return S, det


def geometry(etype, p, xv):
    """Metric terms of one element type.

    Returns dict: xu [N_u,N_e,3] physical solution points, smats [3(alpha),3(i),N_u,N_e]
    (S = |J| J^-1), rcpdjac [N_u,N_e], djac [N_u,N_e], xf [N_f,N_e,3], fnorm [N_f,3,N_e] unit physical
    outward normals, fmag [N_f,N_e] = |S^T n_ref|, affine (bool: J constant in each element).
    """
    ops = refelem.operators(etype, p)
    quadratic = xv.shape[1] in _NQUAD
    if quadratic and _NQUAD[xv.shape[1]] != etype:
        raise ValueError("node count does not match the element type")
    sh = shape2 if quadratic else shape
    Nu, dNu = sh(etype, ops["upts"])
    Nf, dNf = sh(etype, ops["fpts"])
    xu = np.einsum("pv,evi->pei", Nu, xv)
    xf = np.einsum("pv,evi->pei", Nf, xv)
    Ju = np.einsum("pva,evi->peia", dNu, xv)
    S, det = _adjugate(Ju)
    if not np.all(det > 0):
        raise ValueError("non-positive Jacobian in %s elements" % etype)
    Jf = np.einsum("pva,evi->peia", dNf, xv)
    Sf, _ = _adjugate(Jf)
    m = np.einsum("peai,pa->pei", Sf, ops["fnorm"])
    mag = np.sqrt(np.einsum("pei,pei->pe", m, m))
    affine = (etype == "tet" and not quadratic) or bool(np.allclose(Ju, Ju[:1], rtol=0, atol=1e-14 * np.abs(Ju).max()))
    return dict(xu=xu, xf=xf, smats=np.ascontiguousarray(S.transpose(2, 3, 0, 1)), rcpdjac=1.0 / det, djac=det,
                fnorm=np.ascontiguousarray((m / mag[..., None]).transpose(0, 2, 1)), fmag=mag, affine=affine)


# ----------------------------------------------------------------------------- generators
def _grid_vid(idx, dims, periodic):
    """Global vertex id of integer lattice points idx [...,3]; periodic directions wrap."""
    out = np.zeros(idx.shape[:-1], dtype=np.int64)
    for d in range(3):
        c = idx[..., d] % dims[d] if periodic[d] else idx[..., d]
        n = dims[d] if periodic[d] else dims[d] + 1
        out = out * n + c
    return out


_KUHN = []
for _perm in itertools.permutations(range(3)):
    _c = [np.zeros(3, dtype=np.int64)]
    for _a in _perm:
        _e = np.zeros(3, dtype=np.int64)
        _e[_a] = 1
        _c.append(_c[-1] + _e)
    _KUHN.append(np.stack(_c))          # 4 lattice offsets: 0, e_pi0, e_pi0+e_pi1, (1,1,1)
_PRISM_TRIS = [np.array([[0, 0], [1, 0], [1, 1]]), np.array([[0, 0], [1, 1], [0, 1]])]


def _fix_orientation(etype, xv, vid, xref=None, lat=None):
    """Swap two vertices of negatively oriented elements (keeps the vertex set, hence the faces).
    The orientation is read from `xref` (e.g. the unjittered coordinates) when given.  `lat` (the lattice positions of the
    vertices, wanted by `curve_nodes`) is permuted alongside and returned as a third value when given."""
    _, dN = shape(etype, np.zeros((1, 3)))
    J = np.einsum("va,evi->eia", dN[0], xv if xref is None else xref)
    neg = np.linalg.det(J) < 0
    if etype == "tet":
        sw = [0, 1, 3, 2]
    elif etype == "hex":
        sw = [4, 5, 6, 7, 0, 1, 2, 3]
    else:
        sw = [0, 2, 1, 3, 5, 4]
    xv[neg] = xv[neg][:, sw]
    vid[neg] = vid[neg][:, sw]
    if lat is not None:
        lat = lat.astype(np.float64)
        lat[neg] = lat[neg][:, sw]
        return xv, vid, lat
    return xv, vid


def _cells(nx, ny, nz):
    i, j, k = np.meshgrid(np.arange(nx), np.arange(ny), np.arange(nz), indexing="ij")
    return np.stack([i.ravel(), j.ravel(), k.ravel()], axis=1)


def _kuhn_tets(cells, coord_fn, dims, periodic, orient_fn=None, want_lat=False):
    xs, ids, x0, lats = [], [], [], []
    for offs in _KUHN:
        lat = cells[:, None, :] + offs[None, :, :]
        lats.append(lat)
        xs.append(coord_fn(lat))
        if orient_fn is not None:
            x0.append(orient_fn(lat))
        ids.append(_grid_vid(lat, dims, periodic))
    xv = np.stack(xs, axis=1).reshape(-1, 4, 3)
    vid = np.stack(ids, axis=1).reshape(-1, 4)
    xref = np.stack(x0, axis=1).reshape(-1, 4, 3) if orient_fn is not None else None
    return _fix_orientation("tet", xv, vid, xref, np.stack(lats, axis=1).reshape(-1, 4, 3) if want_lat else None)


def _prisms(cells, coord_fn, dims, periodic, tri_axes=(0, 1), ext_axis=2, want_lat=False):
    """Two prisms per lattice cell: triangles in the (tri_axes) plane, extruded along ext_axis."""
    xs, ids, lats = [], [], []
    for tri in _PRISM_TRIS:
        offs = np.zeros((6, 3), dtype=np.int64)
        for lvl in range(2):
            offs[3 * lvl:3 * lvl + 3, tri_axes[0]] = tri[:, 0]
            offs[3 * lvl:3 * lvl + 3, tri_axes[1]] = tri[:, 1]
            offs[3 * lvl:3 * lvl + 3, ext_axis] = lvl
        lat = cells[:, None, :] + offs[None, :, :]
        lats.append(lat)
        xs.append(coord_fn(lat))
        ids.append(_grid_vid(lat, dims, periodic))
    xv = np.stack(xs, axis=1).reshape(-1, 6, 3)
    vid = np.stack(ids, axis=1).reshape(-1, 6)
    return _fix_orientation("pri", xv, vid, None, np.stack(lats, axis=1).reshape(-1, 6, 3) if want_lat else None)


def _hexes(cells, coord_fn, dims, periodic):
    """One hexahedron per lattice cell, vertices in the order of refelem."""
    offs = ((np.array(refelem._VERTS["hex"]) + 1) // 2).astype(np.int64)
    lat = cells[:, None, :] + offs[None, :, :]
    return _fix_orientation("hex", coord_fn(lat).astype(np.float64), _grid_vid(lat, dims, periodic))


def _renumber(mesh, numbering, seed):
    """Element numbering variants: natural, morton (of centroids), random (seeded)."""
    if numbering == "natural":
        return mesh
    rng = np.random.Generator(np.random.PCG64(seed))
    for t in mesh["etypes"]:
        ne = mesh["xv"][t].shape[0]
        if numbering == "random":
            perm = rng.permutation(ne)
        elif numbering == "morton":
            c = mesh["xv"][t].mean(axis=1)
            lo, hi = c.min(0), c.max(0)
            q = ((c - lo) / np.maximum(hi - lo, 1e-300) * 1023.999).astype(np.uint64)
            key = np.zeros(ne, dtype=np.uint64)
            for b in range(10):
                for d in range(3):
                    key |= ((q[:, d] >> np.uint64(b)) & np.uint64(1)) << np.uint64(3 * b + d)
            perm = np.argsort(key, kind="stable")
        else:
            raise ValueError(numbering)
        mesh["xv"][t] = np.ascontiguousarray(mesh["xv"][t][perm])
        mesh["vid"][t] = np.ascontiguousarray(mesh["vid"][t][perm])
        if "xq" in mesh:
            mesh["xq"][t] = np.ascontiguousarray(mesh["xq"][t][perm])
    return mesh


def box_tets(n, length=2 * np.pi, numbering="natural", seed=0):
    """Config 1 (BASELINE.json configs[0]): periodic cube [0,length]^3, n^3 cells, Kuhn 6-tet split."""
    h = length / n
    dims, per = (n, n, n), (True, True, True)
    xv, vid = _kuhn_tets(_cells(n, n, n), lambda lat: lat * h, dims, per)
    m = dict(etypes=["tet"], xv={"tet": xv}, vid={"tet": vid}, period=[length] * 3, bc_tag=None, n=n)
    return _renumber(m, numbering, seed)


def box_hex(n, length=1.0, numbering="natural", seed=0, warp=0.0):
    """Periodic box of n^3 hexahedra (the paper's other mesh type).  warp > 0 displaces the
    interior lattice smoothly (periodic sine field of relative amplitude `warp`), which makes the elements non-affine (trilinear)."""
    h = length / n
    dims, per = (n, n, n), (True, True, True)

    def coord(lat):
        x = lat * h
        if warp > 0:
            k = 2 * np.pi / length
            d = warp * h * np.stack([np.sin(k * x[..., 1]) * np.sin(k * x[..., 2]), np.sin(k * x[..., 0]) * np.sin(k * x[..., 2]),
                                     np.sin(k * x[..., 0]) * np.sin(k * x[..., 1])], axis=-1)
            x = x + d
        return x

    xv, vid = _hexes(_cells(n, n, n), coord, dims, per)
    m = dict(etypes=["hex"], xv={"hex": xv}, vid={"hex": vid}, period=[length] * 3, bc_tag=None, n=n)
    return _renumber(m, numbering, seed)


def _sine_bump(length, amp):
    """x -> x + amp * (periodic sine field): the smooth map the box generators curve their elements with."""
    k = 2 * np.pi / length

    def fn(x):
        d = np.stack([np.sin(k * x[..., 1]) * np.sin(k * x[..., 2]), np.sin(k * x[..., 0]) * np.sin(k * x[..., 2]),
                      np.sin(k * x[..., 0]) * np.sin(k * x[..., 1])], axis=-1)
        return x + amp * d
    return fn


def box_mixed(n, length=1.0, numbering="natural", seed=0, curve=0.0):
    """Config 2 (BASELINE.json configs[1]): periodic box, cells with k < n/2 -> 2 prisms (axis z), others -> 6 tets.
    curve > 0: quadratically curved elements -- the vertices stay, the edge / face / cell nodes of the
    P2 tetrahedra and P2 x P2 prisms follow a smooth periodic displacement field of amplitude `curve` * length."""
    h = length / n
    dims, per = (n, n, n), (True, True, True)
    cells = _cells(n, n, n)
    low = cells[:, 2] < n // 2
    coord = lambda lat: lat * h
    xt, vt = _kuhn_tets(cells[~low], coord, dims, per)
    xp, vp = _prisms(cells[low], coord, dims, per)
    m = dict(etypes=["tet", "pri"], xv={"tet": xt, "pri": xp}, vid={"tet": vt, "pri": vp},
             period=[length] * 3, bc_tag=None, n=n)
    if curve > 0:
        # a fixed smooth map of amplitude A = curve * length: an edge node leaves its chord by ~ (h^2 / 8) |d''| = A pi^2 / (2 n^2),
        # i.e. by (curve pi^2 / (2 n)) h -- the relative curvature vanishes under refinement, as for any smooth geometry
        fn = _sine_bump(length, curve * length)
        m["xq"] = {"tet": curve_nodes("tet", xt, xt, fn), "pri": curve_nodes("pri", xp, xp, fn)}
    return _renumber(m, numbering, seed)


def cylinder_omesh(ntheta=100, nz=15, nlayers=40, nr=40, ratio=1.1, h0=1e-3, jitter=0.15, numbering="natural", seed=0,
                   quadratic=False):
    """Configs 3/5 (BASELINE.json configs[2], [4]): cylinder-like O-mesh, SURVEY D.3 / DESIGN.md reading R19.

    Unit-diameter cylinder at the origin, domain [-9,25]x[-9,9]x[0,pi], span-periodic;
    `nlayers` geometrically stretched prism layers on the wall, then `nr` layers of Kuhn-split tets
    out to the rectangle, seeded vertex jitter in the tet region.  2*ntheta*nz*nlayers prisms,
    6*ntheta*nz*nr tets.  bc tags: 0 = wall (no-slip isothermal), 1 = far field.
    quadratic=True (the paper's cylinder meshes are quadratically curved): same vertices,
    the edge / face nodes of the prisms follow the polar map of the lattice (`curve_nodes`), so the wall is a
    piecewise-quadratic approximation of the circle instead of a polygon; the curvature is blended out linearly across the
    first tetrahedral layer and the far field stays straight-sided.
    """
    rng = np.random.Generator(np.random.PCG64(seed))
    rw = 0.5
    rj = rw + h0 * (ratio ** np.arange(nlayers + 1) - 1) / (ratio - 1)
    rtop = rj[-1]
    nj = nlayers + nr                      # lattice (i, J, k), J = 0..nj
    dims, per = (ntheta, nj, nz), (True, False, True)
    span = np.pi

    def rho_out(th):
        c, s = np.cos(th), np.sin(th)
        with np.errstate(divide="ignore"):
            tx = np.where(c > 0, 25.0 / np.abs(c), 9.0 / np.abs(c))
            ty = 9.0 / np.abs(s)
        return np.minimum(tx, ty)

    # per-vertex jitter table for the tet region interior (indexed by wrapped lattice point)
    jit = np.zeros((ntheta, nj + 1, nz, 3))
    if jitter > 0:
        jit[:, nlayers + 1:nj, :, :] = rng.uniform(-1, 1, size=(ntheta, nr - 1, nz, 3))

    def make_coord(amp):
        def coord(lat):
            i, J, k = lat[..., 0], lat[..., 1], lat[..., 2]
            th = 2 * np.pi * i / ntheta
            ro = rho_out(th)
            jj = np.clip(J - nlayers, 0, nr)
            r_t = rtop + (ro - rtop) * (ratio ** jj - 1) / (ratio ** nr - 1)
            r = np.where(J <= nlayers, rj[np.clip(J, 0, nlayers)], r_t)
            x = np.stack([r * np.cos(th), r * np.sin(th), span * k / nz], axis=-1)
            if amp > 0:
                # local length scale: min of radial, circumferential and spanwise spacing
                jm = np.clip(jj - 1, 0, nr)
                r_m = rtop + (ro - rtop) * (ratio ** jm - 1) / (ratio ** nr - 1)
                lmin = np.minimum(np.minimum(r_t - r_m, r * 2 * np.pi / ntheta), span / nz)
                x = x + amp * lmin[..., None] * jit[i % ntheta, J, k % nz]
            return x
        return coord

    def smooth(lat):
        """The unjittered map for real-valued lattice positions (the wall layers' radii in closed form)."""
        i, J, k = lat[..., 0], lat[..., 1], lat[..., 2]
        th = 2 * np.pi * i / ntheta
        jj = np.clip(J - nlayers, 0, nr)
        r_t = rtop + (rho_out(th) - rtop) * (ratio ** jj - 1) / (ratio ** nr - 1)
        r = np.where(J <= nlayers, rw + h0 * (ratio ** np.minimum(J, nlayers) - 1) / (ratio - 1), r_t)
        return np.stack([r * np.cos(th), r * np.sin(th), span * k / nz], axis=-1)

    cells_p = _cells(ntheta, nlayers, nz)
    cells_t = _cells(ntheta, nr, nz)
    cells_t[:, 1] += nlayers
    amp = jitter
    coord0 = make_coord(0.0)
    xp, vp, lp = _prisms(cells_p, coord0, dims, per, tri_axes=(0, 2), ext_axis=1, want_lat=True)
    _, dN = shape("tet", np.zeros((1, 3)))
    x0, _v = _kuhn_tets(cells_t, coord0, dims, per)
    det0 = np.linalg.det(np.einsum("va,evi->eia", dN[0], x0))
    for _ in range(12):
        # orientation is fixed from the unjittered lattice; halve the jitter until no tet degenerates
        xt, vt, lt = _kuhn_tets(cells_t, make_coord(amp), dims, per, orient_fn=coord0, want_lat=True)
        det = np.linalg.det(np.einsum("va,evi->eia", dN[0], xt))
        if np.all(det > 0.05 * det0):
            break
        amp *= 0.5
    else:
        raise RuntimeError("could not jitter the tet region without inverting elements")

    def bc_tag(cen):
        return np.where(np.hypot(cen[:, 0], cen[:, 1]) < 1.0, 0, 1).astype(np.int32)

    m = dict(etypes=["tet", "pri"], xv={"tet": xt, "pri": xp}, vid={"tet": vt, "pri": vp},
             period=[None, None, span], bc_tag=bc_tag, jitter_amp=amp)
    if quadratic:
        blend = lambda lat: np.clip(nlayers + 1.0 - lat[..., 1], 0.0, 1.0)
        m["xq"] = {"tet": curve_nodes("tet", xt, lt, smooth, blend), "pri": curve_nodes("pri", xp, lp, smooth, blend)}
    return _renumber(m, numbering, seed)


# ----------------------------------------------------------------------------- connectivity
def _face_perm_tables(p):
    """For each vertex permutation of a face, the induced permutation of its flux points.

    tri: weights = barycentric coordinates wrt (A,B,C); quad: bilinear weights wrt (A,B,C,D).
    table[perm][j] = j' such that weights(j')[k] == weights(j)[perm[k]] for all k.
    """
    ops_t = refelem.operators("tet", p)
    sel = ops_t["fface"] == 0
    ab = ops_t["fab"][sel]
    wt = np.stack([1 - (ab[:, 0] + 1) / 2 - (ab[:, 1] + 1) / 2, (ab[:, 0] + 1) / 2, (ab[:, 1] + 1) / 2], axis=1)
    ops_p = refelem.operators("pri", p)
    sel = ops_p["fface"] == 2
    ab = ops_p["fab"][sel]
    a, b = ab[:, 0], ab[:, 1]
    wq = np.stack([(1 - a) * (1 - b), (1 + a) * (1 - b), (1 + a) * (1 + b), (1 - a) * (1 + b)], axis=1) / 4

    def tables(w, perms):
        out = {}
        for perm in perms:
            tgt = w[:, list(perm)]
            d = np.abs(tgt[:, None, :] - w[None, :, :]).max(axis=2)
            j = d.argmin(axis=1)
            if d[np.arange(len(j)), j].max() < 1e-12 and len(set(j.tolist())) == len(j):
                out[perm] = j
        return out

    tri = tables(wt, itertools.permutations(range(3)))
    quad = tables(wq, itertools.permutations(range(4)))
    assert len(tri) == 6 and len(quad) == 8
    return tri, quad


def connectivity(mesh, p, geo=None):
    """Match faces by global vertex ids and pair their flux points.

    Returns (ifaces, bfaces):
      ifaces: dict l_et,l_fpt,l_ele,r_et,r_fpt,r_ele (int32/int32/int64), sorted by (l_et,l_fpt,l_ele);
              L = the side with the smaller (et, ele, face) (reading R9) -- plus nl [3,npairs],
              magl, magr [npairs] when `geo` ({etype: geometry(...)}) is given.
      bfaces: dict tag -> dict et,fpt,ele (+ n [3,nb], mag [nb]) for unmatched faces.
    """
    tri_tab, quad_tab = _face_perm_tables(p)
    ets = mesh["etypes"]
    rec_key, rec_t, rec_e, rec_f, rec_fv = [], [], [], [], []
    foff = {}
    for ti, t in enumerate(ets):
        ops = refelem.operators(t, p)
        vid = mesh["vid"][t]
        ne = vid.shape[0]
        foff[ti] = np.array([np.nonzero(ops["fface"] == f)[0][0] for f in range(len(ops["faces"]))])
        for f, fv in enumerate(ops["faces"]):
            ids = vid[:, list(fv)]
            if len(fv) == 3:
                ids = np.concatenate([ids, np.full((ne, 1), -1, dtype=np.int64)], axis=1)
            rec_fv.append(ids)
            rec_key.append(np.sort(ids, axis=1))
            rec_t.append(np.full(ne, ti, dtype=np.int32))
            rec_e.append(np.arange(ne, dtype=np.int64))
            rec_f.append(np.full(ne, f, dtype=np.int32))
    key = np.concatenate(rec_key)
    ft, fe, ff, fv = (np.concatenate(x) for x in (rec_t, rec_e, rec_f, rec_fv))
    # canonical record order (t, e, f) so that "first of a matched pair" = smaller (et, ele, face)
    order = np.lexsort((ff, fe, ft))
    key, ft, fe, ff, fv = key[order], ft[order], fe[order], ff[order], fv[order]
    srt = np.lexsort((key[:, 3], key[:, 2], key[:, 1], key[:, 0]))   # stable: ties keep (t,e,f) order
    ks = key[srt]
    same = np.all(ks[1:] == ks[:-1], axis=1)
    if np.any(same[1:] & same[:-1]):
        raise ValueError("a face is shared by more than two elements (mesh too small for vertex-id matching?)")
    first = np.nonzero(same)[0]
    li, ri = srt[first], srt[first + 1]
    matched = np.zeros(len(key), dtype=bool)
    matched[li] = True
    matched[ri] = True

    out = {k: [] for k in ("l_et", "l_fpt", "l_ele", "r_et", "r_fpt", "r_ele")}
    is_tri = fv[li][:, 3] < 0
    for tri, tab in ((True, tri_tab), (False, quad_tab)):
        sel = np.nonzero(is_tri == tri)[0]
        if sel.size == 0:
            continue
        nv = 3 if tri else 4
        a, b = fv[li[sel]][:, :nv], fv[ri[sel]][:, :nv]
        perm = (b[:, :, None] == a[:, None, :]).argmax(axis=2)          # b_k = a_perm[k]
        assert np.all(np.take_along_axis(a, perm, axis=1) == b)
        code = np.zeros(len(sel), dtype=np.int64)
        for k in range(nv):
            code = code * 4 + perm[:, k]
        nfp = len(next(iter(tab.values())))
        lut = np.full((4 ** nv, nfp), -1, dtype=np.int64)
        for pm, tbl in tab.items():
            c = 0
            for k in range(nv):
                c = c * 4 + pm[k]
            lut[c] = tbl
        jr = lut[code]
        assert np.all(jr >= 0)
        j = np.arange(nfp)[None, :]
        foff_arr = np.full((len(ets), 8), 0, dtype=np.int64)
        for ti in foff:
            foff_arr[ti, :len(foff[ti])] = foff[ti]
        offl = foff_arr[ft[li[sel]], ff[li[sel]]]
        offr = foff_arr[ft[ri[sel]], ff[ri[sel]]]
        out["l_et"].append(np.repeat(ft[li[sel]], nfp))
        out["l_ele"].append(np.repeat(fe[li[sel]], nfp))
        out["l_fpt"].append((offl[:, None] + j).ravel())
        out["r_et"].append(np.repeat(ft[ri[sel]], nfp))
        out["r_ele"].append(np.repeat(fe[ri[sel]], nfp))
        out["r_fpt"].append((offr[:, None] + jr).ravel())
    ifc = {k: np.concatenate(v) if v else np.zeros(0, dtype=np.int64) for k, v in out.items()}
    o = np.lexsort((ifc["l_ele"], ifc["l_fpt"], ifc["l_et"]))
    ifc = {k: v[o] for k, v in ifc.items()}
    for k in ("l_et", "r_et", "l_fpt", "r_fpt"):
        ifc[k] = ifc[k].astype(np.int32)
    for k in ("l_ele", "r_ele"):
        ifc[k] = ifc[k].astype(np.int64)

    # boundary faces
    bfaces = {}
    bi = np.nonzero(~matched)[0]
    if bi.size:
        if mesh.get("bc_tag") is None:
            raise ValueError("unmatched faces in a mesh without boundary tags")
        cen = np.zeros((bi.size, 3))
        for ti, t in enumerate(ets):
            m = ft[bi] == ti
            if not m.any():
                continue
            fl = refelem.operators(t, p)["faces"]
            xv = mesh["xv"][t]
            for f, fvl in enumerate(fl):
                mm = m & (ff[bi] == f)
                cen[mm] = xv[fe[bi][mm]][:, list(fvl)].mean(axis=1)
        tags = mesh["bc_tag"](cen)
        foff_arr = np.full((len(ets), 8), 0, dtype=np.int64)
        for ti in foff:
            foff_arr[ti, :len(foff[ti])] = foff[ti]
        for tag in np.unique(tags):
            s = bi[tags == tag]
            nfpf = np.where(fv[s][:, 3] < 0, len(next(iter(tri_tab.values()))), len(next(iter(quad_tab.values()))))
            et = np.repeat(ft[s], nfpf)
            el = np.repeat(fe[s], nfpf)
            base = np.repeat(foff_arr[ft[s], ff[s]], nfpf)
            within = np.concatenate([np.arange(k) for k in nfpf]) if s.size else np.zeros(0, dtype=np.int64)
            fpt = base + within
            o = np.lexsort((el, fpt, et))
            bfaces[int(tag)] = dict(et=et[o].astype(np.int32), fpt=fpt[o].astype(np.int32), ele=el[o].astype(np.int64))

    if geo is not None:
        attach_face_geometry(mesh, ifc, bfaces, geo)
    return ifc, bfaces


def attach_face_geometry(mesh, ifc, bfaces, geo):
    ets = mesh["etypes"]
    npairs = len(ifc["l_et"])
    nl = np.zeros((3, npairs))
    magl, magr = np.zeros(npairs), np.zeros(npairs)
    for ti, t in enumerate(ets):
        g = geo[t]
        m = ifc["l_et"] == ti
        nl[:, m] = g["fnorm"][ifc["l_fpt"][m], :, ifc["l_ele"][m]].T
        magl[m] = g["fmag"][ifc["l_fpt"][m], ifc["l_ele"][m]]
        m = ifc["r_et"] == ti
        magr[m] = g["fmag"][ifc["r_fpt"][m], ifc["r_ele"][m]]
    ifc.update(nl=nl, magl=magl, magr=magr)
    for tag, b in bfaces.items():
        nb = len(b["et"])
        n, mag = np.zeros((3, nb)), np.zeros(nb)
        for ti, t in enumerate(ets):
            g = geo[t]
            m = b["et"] == ti
            n[:, m] = g["fnorm"][b["fpt"][m], :, b["ele"][m]].T
            mag[m] = g["fmag"][b["fpt"][m], b["ele"][m]]
        b.update(n=n, mag=mag)


def connectivity_by_coords(mesh, p, geo, tol=1e-9):
    """Independent (slow) pairing by physical flux-point coordinates with periodic wrap -- used to
    check `connectivity` and for meshes too small for vertex-id matching (n < 3).  Fully periodic only."""
    from scipy.spatial import cKDTree
    ets = mesh["etypes"]
    pts, lab = [], []
    for ti, t in enumerate(ets):
        xf = geo[t]["xf"]
        nf, ne, _ = xf.shape
        pts.append(xf.reshape(-1, 3))
        s, e = np.meshgrid(np.arange(nf), np.arange(ne), indexing="ij")
        lab.append(np.stack([np.full(nf * ne, ti), e.ravel(), s.ravel()], axis=1))
    pts, lab = np.concatenate(pts), np.concatenate(lab)
    box = np.array([L for L in mesh["period"]], dtype=np.float64)
    pw = np.mod(pts, box)
    pw[pw >= box - 1e-12] = 0.0
    tree = cKDTree(pw, boxsize=box)
    h = box.min()
    pairs = tree.query_pairs(tol * h, output_type="ndarray")
    cnt = np.bincount(pairs.ravel(), minlength=len(pts))
    if not np.all(cnt == 1):
        raise ValueError("flux points are not paired exactly once")
    a, b = pairs[:, 0], pairs[:, 1]
    ka = lab[a, 0] * (1 << 40) + lab[a, 1] * 1024 + lab[a, 2]
    kb = lab[b, 0] * (1 << 40) + lab[b, 1] * 1024 + lab[b, 2]
    sw = kb < ka
    a, b = np.where(sw, b, a), np.where(sw, a, b)
    ifc = dict(l_et=lab[a, 0].astype(np.int32), l_ele=lab[a, 1].astype(np.int64), l_fpt=lab[a, 2].astype(np.int32),
               r_et=lab[b, 0].astype(np.int32), r_ele=lab[b, 1].astype(np.int64), r_fpt=lab[b, 2].astype(np.int32))
    o = np.lexsort((ifc["l_ele"], ifc["l_fpt"], ifc["l_et"]))
    ifc = {k: v[o] for k, v in ifc.items()}
    attach_face_geometry(mesh, ifc, {}, geo)
    return ifc, {}
