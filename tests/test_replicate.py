"""`fr_inputs.cases.replicate` (the size-up of the sustained run, BASELINE.json configs[4]): K disjoint copies as one case.
CPU: the oracle on the replica equals the oracle on each copy's own state (the copies do not touch).  GPU: the library on the
replica, compact metric terms included, equals the oracle."""
import numpy as np
import pytest

from fr_inputs import cases, state
from util import oracle_rhs


def _small(system="ns"):
    return cases.config3(p=2, ntheta=12, nz=3, nlayers=3, nr=3, numbering="random", system=system)


def test_replica_oracle_equals_per_copy_oracle():
    case = _small()
    K = 3
    rep = cases.replicate(case, K, amp=0.005, seed=11)
    ne = [e["neles"] for e in case["eles"]]
    assert [e["neles"] for e in rep["eles"]] == [K * n for n in ne]
    assert len(rep["ifc"]["l_ele"]) == K * len(case["ifc"]["l_ele"])
    # every flux point of the replica appears exactly once among pairs and boundary lists
    for t, e in enumerate(rep["eles"]):
        cnt = np.zeros((e["nfpts"], e["neles"]), dtype=np.int64)
        for s in ("l", "r"):
            m = rep["ifc"][s + "_et"] == t
            np.add.at(cnt, (rep["ifc"][s + "_fpt"][m], rep["ifc"][s + "_ele"][m]), 1)
        for b in rep["bcs"]:
            m = b["et"] == t
            np.add.at(cnt, (b["fpt"][m], b["ele"][m]), 1)
        assert (cnt == 1).all()
    full = oracle_rhs(rep)
    for k in range(K):
        one = dict(case)
        one["u0"] = [u[:, :, k * n:(k + 1) * n] for u, n in zip(rep["u0"], ne)]
        ref = oracle_rhs(one)
        for f, r, n in zip(full, ref, ne):
            assert np.array_equal(f[:, :, k * n:(k + 1) * n], r)
    # copy 0 keeps the case's state, the others differ from it
    assert np.array_equal(rep["u0"][0][:, :, :ne[0]], case["u0"][0])
    assert not np.array_equal(rep["u0"][0][:, :, ne[0]:2 * ne[0]], case["u0"][0])


def test_replica_compact_keeps_what_setup_reads():
    case = _small("euler")
    a, b = cases.replicate(case, 2), cases.replicate(case, 2, compact=True)
    for ea, eb in zip(a["eles"], b["eles"]):
        if ea["affine"]:
            assert eb["smats"].shape[2] == 1 and eb["rcpdjac"].shape[0] == 1
            assert np.array_equal(ea["smats"][:, :, 0, :], eb["smats"][:, :, 0, :])
            assert np.array_equal(ea["rcpdjac"][0, :], eb["rcpdjac"][0, :])
        else:
            assert np.array_equal(ea["smats"], eb["smats"])
        assert eb["xu"] is None
    with pytest.raises(ValueError):
        cases.replicate(case, 0)


@pytest.mark.gpu
@pytest.mark.parametrize("prec,tol", [("f64", 1e-11), ("f32", 2e-5)])
def test_gpu_replica_matches_oracle(prec, tol):
    from gpu_util import gpu_rhs, round_case_to_f32
    from paper_1409_0405_b200 import Context
    case = _small()
    rep = cases.replicate(case, 3, amp=0.005, seed=11)
    if prec == "f32":
        rep = round_case_to_f32(rep)
    ref = oracle_rhs(rep)
    comp = cases.replicate(case, 3, compact=True)
    ctx = Context(comp, prec=prec, stepper="rk45")
    got, _ = gpu_rhs(ctx, rep["u0"])
    ctx.close()
    num, den = np.zeros(5), np.zeros(5)
    for g, r in zip(got, ref):
        num = np.maximum(num, np.abs(g - r).max(axis=(0, 2)))
        den = np.maximum(den, np.abs(r).max(axis=(0, 2)))
    assert (num / den).max() < tol


def _totals(case, us):
    """quadrature-weighted sums of the five conserved variables over all elements (omega_j |J| u), FP64"""
    tot = np.zeros(5)
    for e, u in zip(case["eles"], us):
        w = e["wts"][:, None] * e["djac"]
        tot += (w[:, None, :] * u).sum(axis=(0, 2))
    return tot


@pytest.mark.gpu
@pytest.mark.parametrize("prec", ["f64", "f32"])
def test_gpu_ten_step_prefix_drift_matches_oracle(prec):
    """BASELINE.json configs[4]: "energy/conservation drift against the oracle on a 10-step prefix".  The sustained run's
    recipe (config-3 generator, p = 3, replicated copies with their own perturbations, compact metric terms, RK45[2R+] graph
    replay with fixed dt) at a size the oracle steps in seconds: the change of the conserved totals over 10 steps and the
    state itself against the oracle's ten rk45_step calls."""
    from gpu_util import round_case_to_f32
    from oracle import fr_oracle as O
    from paper_1409_0405_b200 import Context
    case = cases.config3(p=3, ntheta=12, nz=3, nlayers=3, nr=3, numbering="random")
    rep = cases.replicate(case, 2, amp=0.005, seed=cases.SEEDS["c5"])
    comp = cases.replicate(case, 2, amp=0.005, seed=cases.SEEDS["c5"], compact=True)
    c = round_case_to_f32(rep) if prec == "f32" else rep
    f = lambda us: O.rhs(c["cfg"], c["eles"], c["ifc"], c["bcs"], us)
    dt, nsteps = 4e-6, 10                         # the sustained run's dt (the wall layers do not allow 2e-5 at p = 3)
    ref = c["u0"]
    for _ in range(nsteps):
        ref = O.rk45_step(f, ref, dt)
    ctx = Context(comp, prec=prec, stepper="rk45")
    ctx.set_state(rep["u0"])
    ctx.rk_run(dt, nsteps)
    ctx.sync()
    got = ctx.get_state()
    ctx.close()
    assert all(np.isfinite(g).all() for g in got)
    t0, tr, tg = _totals(rep, c["u0"]), _totals(rep, ref), _totals(rep, got)
    scale = np.abs(t0).max()
    drift_ref, drift_got = (tr - t0) / scale, (tg - t0) / scale
    assert np.abs(drift_ref).max() > 2e-8          # open boundaries: the totals do move, so the comparison is not 0 = 0
    # FP64: the drift itself agrees to 1e-9 of its size.  FP32: 50 stage updates of an FP32 state round the totals by a few
    # 2^-24 relative (the sums are taken in FP64 on the host from the FP32 state)
    tol = 1e-9 * np.abs(drift_ref).max() if prec == "f64" else 5e-7
    assert np.abs(drift_got - drift_ref).max() <= tol, (drift_got, drift_ref)
    num = max(np.abs(a - b).max() for a, b in zip(got, ref))
    den = max(np.abs(b).max() for b in ref)
    assert num / den <= (1e-11 if prec == "f64" else 2e-6)
