"""Shared helpers for the tests (no method arithmetic)."""
import numpy as np


def field_errors(got, ref, joint_momentum=False):
    """Max-norm relative error per conserved variable, jointly over element types (reading R16):
    err_k = max |got - ref| / max |ref| over all types, points and elements, for variable k.
    joint_momentum: the three momentum components are one vector field and share the denominator max_k max |ref_k| -- a component
    that vanishes by symmetry (rho v_z of a z-invariant flow) has no scale of its own."""
    num, den = np.zeros(5), np.zeros(5)
    for g, r in zip(got, ref):
        num = np.maximum(num, np.abs(g - r).max(axis=(0, 2)))
        den = np.maximum(den, np.abs(r).max(axis=(0, 2)))
    if joint_momentum:
        den = den.copy()
        den[1:4] = den[1:4].max()
    return num / np.maximum(den, 1e-300), den


def conservation_defect(case, dudt):
    """sum_types sum_e sum_rho omega_rho |J| dudt, relative to the same sum of absolute values (T2)."""
    tot, ab = np.zeros(5), np.zeros(5)
    for e, d in zip(case["eles"], dudt):
        w = e["wts"][:, None, None] * e["djac"][:, None, :]
        tot += (w * d).sum(axis=(0, 2))
        ab += np.abs(w * d).sum(axis=(0, 2))
    return tot / np.maximum(ab, 1e-300)


def oracle_rhs(case, us=None):
    from oracle import fr_oracle
    return fr_oracle.rhs(case["cfg"], case["eles"], case["ifc"], case["bcs"], case["u0"] if us is None else us)


EPS32 = 2.0 ** -24


def oracle_rhs_with_amplification(case, us=None, joint_momentum=False):
    """Oracle RHS plus the a-priori round-off amplification of its last step per variable (reading R23):
    amp_k = max (|M132| |F~| + |M3| |D|) / |J|  divided by  max |dudt_k|.  A computation that stores F~ and D in a
    precision with unit round-off eps cannot be closer to the exact result than ~ eps * amp_k."""
    from oracle import fr_oracle
    parts = {}
    ref = fr_oracle.rhs(case["cfg"], case["eles"], case["ifc"], case["bcs"], case["u0"] if us is None else us, parts)
    A, den = np.zeros(5), np.zeros(5)
    for e, ft, d, r in zip(case["eles"], parts["ftil"], parts["d"], ref):
        nu = e["nupts"]
        a = (np.abs(e["M132"]) @ np.abs(ft.reshape(3 * nu, -1)) + np.abs(e["M3"]) @ np.abs(d.reshape(d.shape[0], -1)))
        a = a.reshape(r.shape) * e["rcpdjac"][:, None, :]
        A = np.maximum(A, a.max(axis=(0, 2)))
        den = np.maximum(den, np.abs(r).max(axis=(0, 2)))
    if joint_momentum:
        A[1:4] = A[1:4].max()
        den[1:4] = den[1:4].max()
    return ref, A / np.maximum(den, 1e-300)
