"""Pins for the time steppers of the oracle: exact order conditions of RK45[2R+] (the coefficients are
not printed in the paper -- PAPER.md:116 names the scheme, reading R12) and empirical convergence slopes."""
from fractions import Fraction

import numpy as np

from oracle import fr_oracle as O


def _butcher():
    a = [Fraction(n, d) for n, d in O.RK45_A_FRAC]
    b = [Fraction(n, d) for n, d in O.RK45_B_FRAC]
    A = [[Fraction(0)] * 5 for _ in range(5)]
    for i in range(1, 5):
        for j in range(i):
            A[i][j] = a[j] if j == i - 1 else b[j]          # 2R van der Houwen form
    c = [sum(r) for r in A]
    return A, b, c


def test_rk45_order_conditions_exact():
    A, b, c = _butcher()
    dot = lambda x, y: sum(p * q for p, q in zip(x, y))
    Ac = [dot(r, c) for r in A]
    Ac2 = [dot(r, [ci * ci for ci in c]) for r in A]
    AAc = [dot(r, Ac) for r in A]
    conds = [(sum(b), 1), (dot(b, c), Fraction(1, 2)), (dot(b, [x * x for x in c]), Fraction(1, 3)),
             (dot(b, Ac), Fraction(1, 6)), (dot(b, [x ** 3 for x in c]), Fraction(1, 4)),
             (dot(b, [x * y for x, y in zip(c, Ac)]), Fraction(1, 8)), (dot(b, Ac2), Fraction(1, 12)),
             (dot(b, AAc), Fraction(1, 24))]
    for got, want in conds:
        assert abs(float(got - want)) < 1e-24
    assert [float(x) for x in O.RK45_A] == [float(Fraction(n, d)) for n, d in O.RK45_A_FRAC]
    assert [float(x) for x in O.RK45_B] == [float(Fraction(n, d)) for n, d in O.RK45_B_FRAC]


def test_rk_slopes_on_linear_ode():
    lam = -1.3 + 0.7j
    f = lambda us: [lam * u for u in us]
    for step, order in ((O.euler_step, 1), (O.rk4_step, 4), (O.rk45_step, 4)):
        errs = []
        for n in (8, 16, 32):
            u = [np.array([1.0 + 0j])]
            for _ in range(n):
                u = step(f, u, 1.0 / n)
            errs.append(abs(u[0][0] - np.exp(lam)))
        slopes = np.log2(np.array(errs[:-1]) / np.array(errs[1:]))
        assert np.all(slopes > order - 0.3) and np.all(slopes < order + 0.6), slopes


def test_rk4_matches_stability_polynomial():
    # one RK4 step on u' = lam u is exactly the degree-4 Taylor polynomial of exp(lam dt)
    z = 0.3 - 0.2j
    u = O.rk4_step(lambda us: [z * x for x in us], [np.array([1.0 + 0j])], 1.0)[0][0]
    assert abs(u - (1 + z + z ** 2 / 2 + z ** 3 / 6 + z ** 4 / 24)) < 1e-15
    # RK45: a 5-stage 4th-order scheme matches the Taylor polynomial through z^4
    u5 = O.rk45_step(lambda us: [z * x for x in us], [np.array([1.0 + 0j])], 1.0)[0][0]
    assert abs(u5 - np.exp(z)) < 2 * abs(z) ** 5 / 120
