"""Pins for the synthetic meshes, metric terms and flux-point connectivity (inputs of both sides)."""
import numpy as np
import pytest

from fr_inputs import cases, mesh as M, refelem as R


def _geo(m, p):
    return {t: M.geometry(t, p, m["xq"][t] if "xq" in m else m["xv"][t]) for t in m["etypes"]}


MESHES = {
    "tets4": lambda: M.box_tets(4),
    "mixed4": lambda: M.box_mixed(4),
    "mixed4_random": lambda: M.box_mixed(4, numbering="random", seed=3),
    "cyl": lambda: M.cylinder_omesh(ntheta=16, nz=4, nlayers=5, nr=5, seed=11),
    "hex3_warped": lambda: M.box_hex(3, numbering="random", seed=5, warp=0.12),
    "mixed4_curved": lambda: M.box_mixed(4, numbering="random", seed=3, curve=0.08),
    "cyl_curved": lambda: M.cylinder_omesh(ntheta=16, nz=4, nlayers=5, nr=5, seed=11, quadratic=True),
}


@pytest.mark.parametrize("name", list(MESHES))
@pytest.mark.parametrize("p", [1, 3])
def test_pairs_cover_every_flux_point_once_and_coincide(name, p):
    m = MESHES[name]()
    geo = _geo(m, p)
    ifc, bf = M.connectivity(m, p, geo)
    seen = {ti: np.zeros((R.operators(t, p)["nfpts"], m["xv"][t].shape[0]), dtype=int) for ti, t in enumerate(m["etypes"])}
    for s in ("l", "r"):
        for ti in seen:
            k = ifc[s + "_et"] == ti
            np.add.at(seen[ti], (ifc[s + "_fpt"][k], ifc[s + "_ele"][k]), 1)
    for b in bf.values():
        for ti in seen:
            k = b["et"] == ti
            np.add.at(seen[ti], (b["fpt"][k], b["ele"][k]), 1)
    assert all(np.all(v == 1) for v in seen.values())
    # physical coordinates of paired points coincide (modulo the period); normals are opposite
    n = len(ifc["l_et"])
    xl, xr, nr, wl, wr = np.zeros((n, 3)), np.zeros((n, 3)), np.zeros((n, 3)), np.zeros(n), np.zeros(n)
    for ti, t in enumerate(m["etypes"]):
        g, fw = geo[t], R.operators(t, p)["fwts"]
        k = ifc["l_et"] == ti
        xl[k] = g["xf"][ifc["l_fpt"][k], ifc["l_ele"][k]]
        wl[k] = fw[ifc["l_fpt"][k]]
        k = ifc["r_et"] == ti
        xr[k] = g["xf"][ifc["r_fpt"][k], ifc["r_ele"][k]]
        nr[k] = g["fnorm"][ifc["r_fpt"][k], :, ifc["r_ele"][k]]
        wr[k] = fw[ifc["r_fpt"][k]]
    d = xl - xr
    for a in range(3):
        if m["period"][a]:
            d[:, a] -= m["period"][a] * np.round(d[:, a] / m["period"][a])
    assert np.abs(d).max() < 1e-12
    assert np.abs(ifc["nl"].T + nr).max() < 1e-10
    # mag_L w_L = mag_R w_R: both sides integrate the same physical face
    assert np.abs(ifc["magl"] * wl - ifc["magr"] * wr).max() < 1e-12 * np.abs(ifc["magl"] * wl).max()
    # L is the side with the smaller (et, ele); pairs sorted by (l_et, l_fpt, l_ele)
    assert np.all((ifc["l_et"] < ifc["r_et"]) | ((ifc["l_et"] == ifc["r_et"]) & (ifc["l_ele"] <= ifc["r_ele"])))
    key = (ifc["l_et"].astype(np.int64) << 50) + (ifc["l_fpt"].astype(np.int64) << 40) + ifc["l_ele"]
    assert np.all(np.diff(key) > 0)


@pytest.mark.parametrize("name", ["tets4", "mixed4", "mixed4_curved"])
def test_vertex_pairing_equals_coordinate_pairing(name):
    m = MESHES[name]()
    geo = _geo(m, 2)
    a, _ = M.connectivity(m, 2, geo)
    b, _ = M.connectivity_by_coords(m, 2, geo)
    for k in a:
        assert np.array_equal(a[k], b[k]) if a[k].dtype.kind == "i" else np.allclose(a[k], b[k], atol=1e-14)


@pytest.mark.parametrize("name", list(MESHES))
def test_closed_elements_and_volume(name):
    p = 2
    m = MESHES[name]()
    geo = _geo(m, p)
    vol = 0.0
    for t in m["etypes"]:
        o, g = R.operators(t, p), geo[t]
        # sum over flux points of w * mag * n = integral of the outward normal over a closed surface = 0
        closed = np.einsum("f,fe,fie->ie", o["fwts"], g["fmag"], g["fnorm"])
        h2 = (np.einsum("f,fe->e", o["fwts"], g["fmag"]))
        assert np.abs(closed).max() < 1e-12 * h2.max()
        vol += (o["wts"][:, None] * g["djac"]).sum()
        assert np.allclose(g["smats"][:, :, :, 0].transpose(2, 0, 1) @ np.linalg.inv(g["smats"][:, :, :, 0].transpose(2, 0, 1)),
                           np.eye(3)[None], atol=1e-12)
    if name == "tets4":
        assert abs(vol - (2 * np.pi) ** 3) < 1e-11 * vol
    if name.startswith("mixed"):
        assert abs(vol - 1.0) < 1e-13
    if name == "cyl":
        # straight-sided O-mesh: volume = (outer polygon through the rectangle - inner 16-gon) x span pi
        nth = 16
        th = 2 * np.pi * np.arange(nth) / nth
        c, s_ = np.cos(th), np.sin(th)
        with np.errstate(divide="ignore"):
            ro = np.minimum(np.where(c > 0, 25.0, 9.0) / np.abs(c), 9.0 / np.abs(s_))
        outer = 0.5 * np.sum(ro * np.roll(ro, -1)) * np.sin(2 * np.pi / nth)
        inner = 0.5 * nth * 0.25 * np.sin(2 * np.pi / nth)
        assert abs(vol - (outer - inner) * np.pi) < 1e-10 * vol


def test_config_counts():
    # reading R18: 16^3 cells -> 4096 prisms + 12288 tets
    m = M.box_mixed(16)
    assert m["xv"]["pri"].shape[0] == 4096 and m["xv"]["tet"].shape[0] == 12288
    c = cases.config1()
    assert c["eles"][0]["neles"] == 384 and c["eles"][0]["nupts"] == 10 and len(c["ifc"]["l_et"]) == 4608
    assert cases.ndof(c) == 3840


def test_cylinder_bc_lists():
    m = M.cylinder_omesh(ntheta=16, nz=4, nlayers=5, nr=5, seed=11)
    p = 2
    geo = _geo(m, p)
    _, bf = M.connectivity(m, p, geo)
    T = 6
    assert len(bf[0]["et"]) == 2 * 16 * 4 * T and len(bf[1]["et"]) == 2 * 16 * 4 * T
    assert np.all(bf[0]["et"] == 1) and np.all(bf[1]["et"] == 0)      # wall on prisms, far field on tets
    # wall normals point towards the axis, far-field normals away from it
    xw = geo["pri"]["xf"][bf[0]["fpt"], bf[0]["ele"]]
    assert np.all(np.einsum("in,ni->n", bf[0]["n"][:2], xw[:, :2]) < 0)
    xo = geo["tet"]["xf"][bf[1]["fpt"], bf[1]["ele"]]
    assert np.all(np.einsum("in,ni->n", bf[1]["n"][:2], xo[:, :2]) > 0)


# ---------------------------------------------------------------------------- quadratic geometry
@pytest.mark.parametrize("etype", ["tet", "pri", "hex"])
def test_quadratic_shape_functions(etype):
    """Nodal on `quad_nodes` (vertices first), partition of unity, exact on the element's quadratic space, and equal to the linear
    shape functions' map when the nodes sit on a straight element."""
    q = M.quad_nodes(etype)
    nv = len(R._VERTS[etype])
    assert q.shape == ({"tet": 10, "pri": 18, "hex": 27}[etype], 3)
    assert np.array_equal(q[:nv], np.array(R._VERTS[etype], dtype=float))
    N, dN = M.shape2(etype, q)
    assert np.abs(N - np.eye(len(q))).max() < 1e-13
    rng = np.random.Generator(np.random.PCG64(5))
    x = rng.uniform(-0.9, -0.1, (7, 3))
    N, dN = M.shape2(etype, x)
    assert np.abs(N.sum(1) - 1).max() < 1e-13 and np.abs(dN.sum(1)).max() < 1e-12
    f = lambda y: 0.3 + y[:, 0] - 2 * y[:, 2] + y[:, 0] * y[:, 1] - 0.5 * y[:, 2] ** 2 + 0.25 * y[:, 1] * y[:, 2]
    df = lambda y: np.stack([1 + y[:, 1], y[:, 0] + 0.25 * y[:, 2], -2 - y[:, 2] + 0.25 * y[:, 1]], axis=1)
    assert np.abs(N @ f(q) - f(x)).max() < 1e-13
    assert np.abs(np.einsum("pqa,q->pa", dN, f(q)) - df(x)).max() < 1e-12
    # straight element: quadratic nodes at the linear map of the reference nodes reproduce the linear geometry
    xv = rng.uniform(-1, 1, (1, nv, 3)) * 0.2 + np.array(R._VERTS[etype], dtype=float)[None]
    Nl, dNl = M.shape(etype, q)
    xq = np.einsum("qv,evi->eqi", Nl, xv)
    Nlx, dNlx = M.shape(etype, x)
    assert np.abs(np.einsum("pq,eqi->epi", N, xq) - np.einsum("pv,evi->epi", Nlx, xv)).max() < 1e-13
    assert np.abs(np.einsum("pqa,eqi->epia", dN, xq) - np.einsum("pva,evi->epia", dNlx, xv)).max() < 1e-12


def test_curved_cylinder_converges_to_the_circle_at_fourth_order():
    """The straight-sided O-mesh approximates the wall by a polygon (volume / area errors O(h^2)); with quadratic elements the
    prism layer's volume and the wall's area converge at fourth order to pi (r_top^2 - r_w^2) * span and 2 pi r_w * span."""
    nl = 3
    rtop = 0.5 + 1e-3 * (1.1 ** nl - 1) / 0.1
    vol_exact, area_exact = np.pi * (rtop ** 2 - 0.25) * np.pi, 2 * np.pi * 0.5 * np.pi
    err = {}
    for quad in (False, True):
        for nth in (12, 24):
            c = cases.config3(p=3, ntheta=nth, nz=3, nlayers=nl, nr=3, numbering="random", quadratic=quad)
            e = [e for e in c["eles"] if e["etype"] == "pri"][0]
            assert e["affine"] is False and c["eles"][0]["affine"] is (not quad)
            vol = (e["wts"][:, None] * e["djac"]).sum()
            wall = [b for b in c["bcs"] if b["type"] == "wall"][0]
            area = sum((c["eles"][t]["fwts"][wall["fpt"][wall["et"] == t]] * wall["mag"][wall["et"] == t]).sum()
                       for t in range(len(c["eles"])))
            err[quad, nth] = (abs(vol / vol_exact - 1), abs(area / area_exact - 1))
    for k in (0, 1):
        assert 3.5 < err[False, 12][k] / err[False, 24][k] < 4.5          # second order
        assert 13.0 < err[True, 12][k] / err[True, 24][k] < 19.0          # fourth order
        assert err[True, 24][k] < 2e-5 and err[False, 24][k] > 2e-3
