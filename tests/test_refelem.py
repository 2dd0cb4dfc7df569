"""Pins for the operator matrices / point sets handed to both the oracle and fr_setup.

Table 2 of the paper fixes the shapes; everything else is fixed by the mathematics:
an operator that is exact on the whole polynomial space of a unisolvent point set is unique, so the
polynomial-exactness checks (I1, I2) pin M0, M1, M2, M4 completely, and the lifting identities
(I3-I6) pin M3 and M6.  A transposed operand, wrong sign or dropped area factor fails here.
"""
import itertools

import numpy as np
import pytest

from fr_inputs import refelem as R

CASES = [(t, p) for t in ("tet", "pri", "hex") for p in (1, 2, 3, 4)]
# Table 2, PAPER.md:43-50 ("dim M0", printed as N_u x N_f; reading R1: M0 is N_f x N_u)
def _load_table2():
    """Table 2 of the paper, kept as a cited text fixture."""
    import os
    out = {}
    with open(os.path.join(os.path.dirname(__file__), "golden", "table2_m0_dims.txt")) as f:
        for line in f:
            if line.strip() and not line.startswith("#"):
                t, p_, nu, nf = line.split()
                out[(t, int(p_))] = (int(nu), int(nf))
    return out


TABLE2 = _load_table2()


def _space(etype, p):
    rng = range(p + 1)
    if etype == "tet":
        return [e for e in itertools.product(rng, rng, rng) if sum(e) <= p]
    if etype == "pri":
        return [e for e in itertools.product(rng, rng, rng) if e[0] + e[1] <= p]
    return list(itertools.product(rng, rng, rng))


def _mono(x, e, d=None):
    out = np.ones(len(x))
    for k in range(3):
        if d == k:
            out = out * (e[k] * x[:, k] ** (e[k] - 1) if e[k] > 0 else 0.0)
        else:
            out = out * x[:, k] ** e[k]
    return out


@pytest.mark.parametrize("etype,p", CASES)
def test_table2_shapes(etype, p):
    o = R.operators(etype, p)
    nu, nf = TABLE2[(etype, p)]
    assert (o["nupts"], o["nfpts"]) == (nu, nf) == R.npts(etype, p)
    assert o["M0"].shape == (nf, nu) and o["M3"].shape == (nu, nf)
    assert o["M132"].shape == (nu, 3 * nu) and o["M460"].shape == (3 * nu, nu) and o["M6"].shape == (3 * nu, nf)


@pytest.mark.parametrize("etype,p", CASES)
def test_I1_I2_polynomial_exactness(etype, p):
    o = R.operators(etype, p)
    nu = o["nupts"]
    xu, xf = o["upts"], o["fpts"]
    for e in _space(etype, p):
        q = _mono(xu, e)
        scale = max(1.0, np.abs(q).max())
        assert np.abs(o["M0"] @ q - _mono(xf, e)).max() < 2e-14 * scale
        g = o["M4"] @ q
        for a in range(3):
            assert np.abs(g[a * nu:(a + 1) * nu] - _mono(xu, e, d=a)).max() < 2e-13 * scale
            # M1 applied to the vector field q * e_a is d_a q ; M2 is n_a * q at the flux points
            f = np.zeros(3 * nu)
            f[a * nu:(a + 1) * nu] = q
            assert np.abs(o["M1"] @ f - _mono(xu, e, d=a)).max() < 2e-13 * scale
            assert np.abs(o["M2"] @ f - o["fnorm"][:, a] * _mono(xf, e)).max() < 2e-14 * scale
    one = np.ones(nu)
    assert np.abs(o["M0"] @ one - 1).max() < 1e-14 and np.abs(o["M4"] @ one).max() < 1e-13


@pytest.mark.parametrize("etype,p", CASES)
def test_I3_to_I6_lifting_identities(etype, p):
    o = R.operators(etype, p)
    nu, nf = o["nupts"], o["nfpts"]
    vol = {"tet": 4.0 / 3.0, "pri": 4.0, "hex": 8.0}[etype]
    assert abs(o["wts"].sum() - vol) < 1e-14
    # face weights sum to the true reference face areas (area factor included)
    V = R.verts(etype)
    for fi, fv in enumerate(o["faces"]):
        A, B, D = V[fv[0]], V[fv[1]], V[fv[-1]]
        area = np.linalg.norm(np.cross(B - A, D - A)) * (0.5 if len(fv) == 3 else 1.0)
        assert abs(o["fwts"][o["fface"] == fi].sum() - area) < 1e-14
    assert np.abs(o["wts"] @ o["M3"] - o["fwts"]).max() < 1e-14                       # I3
    assert np.abs(o["wts"] @ o["M1"] - o["fwts"] @ o["M2"]).max() < 1e-14            # I4 divergence theorem
    rng = np.random.default_rng(5)
    c = rng.standard_normal(3)
    cvec = np.repeat(c, nu)
    assert np.abs(o["M132"] @ cvec + o["M3"] @ (o["fnorm"] @ c)).max() < 1e-13       # I5
    for a in range(3):                                                               # I6
        assert np.array_equal(o["M6"][a * nu:(a + 1) * nu], o["M3"] * o["fnorm"][None, :, a]) or \
            np.abs(o["M6"][a * nu:(a + 1) * nu] - o["M3"] * o["fnorm"][None, :, a]).max() < 1e-15
    assert np.abs(o["M132"] - (o["M1"] - o["M3"] @ o["M2"])).max() < 1e-13
    assert np.abs(o["M460"] - (o["M4"] - o["M6"] @ o["M0"])).max() < 1e-13
    # weighted integration by parts with the lift: for polynomials q, phi in the space,
    #   int phi (M3 g) = int_face phi g  (definition of the DG correction, reading R7) -> tested against B built here
    # via: wts-weighted exactness of products is not available (wts is not a degree-2p rule), so use I3..I5 only.


@pytest.mark.parametrize("p", [1, 2, 3, 4, 5, 6])
def test_point_sets_interior_and_symmetric(p):
    o = R.operators("tet", p) if p <= 4 else None
    with R.mp.workdps(30):
        tri = np.array([[float(c) for c in pt] for pt in R._tri_pts_mp(p)])
        tet = np.array([[float(c) for c in pt] for pt in R._tet_pts_mp(p)])
    lam3 = np.stack([-(tri[:, 0] + tri[:, 1]) / 2, (1 + tri[:, 0]) / 2, (1 + tri[:, 1]) / 2], 1)
    lam4 = np.stack([-(1 + tet.sum(1)) / 2, (1 + tet[:, 0]) / 2, (1 + tet[:, 1]) / 2, (1 + tet[:, 2]) / 2], 1)
    assert lam3.min() > 0.01 and lam4.min() > 0.01
    for lam in (lam3, lam4):
        for perm in itertools.permutations(range(lam.shape[1])):
            d = np.abs(lam[:, list(perm)][:, None, :] - lam[None, :, :]).max(axis=2)
            assert d.min(axis=1).max() < 1e-13          # the set is invariant under vertex permutations
    if o is not None:
        assert np.abs(o["M0"]).sum(axis=1).max() < 4.0  # well-conditioned interpolation (matters for FP32)
