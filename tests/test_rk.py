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


# ---------------------------------------------------------------------------- embedded pair and step-size control (NEXT-3)
def test_rk45_embedded_weights_are_third_order_exactly():
    A, b, c = _butcher()
    bh = [Fraction(n, d) for n, d in O.RK45_BHAT_FRAC]
    dot = lambda x, y: sum(p * q for p, q in zip(x, y))
    Ac = [dot(r, c) for r in A]
    for got, want in ((sum(bh), 1), (dot(bh, c), Fraction(1, 2)), (dot(bh, [x * x for x in c]), Fraction(1, 3)),
                      (dot(bh, Ac), Fraction(1, 6))):
        assert abs(float(got - want)) < 1e-24
    # ... and not fourth order (otherwise the difference would not estimate the local error)
    assert abs(float(dot(bh, [x ** 3 for x in c]) - Fraction(1, 4))) > 1e-3
    assert [float(x) for x in O.RK45_BHAT] == [float(Fraction(n, d)) for n, d in O.RK45_BHAT_FRAC]


def test_embedded_error_estimate():
    """u' = lam u: E = (R(z) - Rhat(z)) u with R - Rhat = O(z^4); the estimate follows dt^4 and the step equals rk45_step."""
    lam = -0.9 + 0.4j
    f = lambda us: [lam * u for u in us]
    u0 = [np.array([1.0 + 0.5j, -2.0 + 0j])]
    es = []
    for dt in (0.2, 0.1, 0.05):
        X, E = O.rk45_step_with_error(f, u0, dt)
        assert np.array_equal(X[0], O.rk45_step(f, u0, dt)[0])
        es.append(np.abs(E[0]).max())
        # third-order solution u+ - E matches exp(z) to O(z^4), the fourth-order one to O(z^5)
        z = lam * dt
        assert np.abs((X[0] - E[0]) / u0[0] - np.exp(z)).max() < 2 * abs(z) ** 4
        assert np.abs(X[0] / u0[0] - np.exp(z)).max() < abs(z) ** 5
    slopes = np.log2(np.array(es[:-1]) / np.array(es[1:]))
    assert np.all(np.abs(slopes - 4) < 0.25), slopes


def test_error_norm_and_pi_factor_closed_forms():
    E = [np.array([[3e-6, -4e-6]]), np.array([[0.0]])]
    a = [np.array([[1.0, -2.0]]), np.array([[5.0]])]
    b = [np.array([[-3.0, 1.0]]), np.array([[5.0]])]
    # scales: 1e-6 + 1e-6 * (3, 2, 5)  ->  (3e-6/4e-6)^2 + (4e-6/3e-6)^2 + 0 over 3 entries
    want = np.sqrt(((3 / 4) ** 2 + (4 / 3) ** 2) / 3)
    assert abs(O.error_norm(E, a, b, 1e-6, 1e-6) - want) < 1e-15
    assert abs(O.pi_factor(0.5, 1.0) - 0.8 * 0.5 ** -0.175) < 1e-15
    assert abs(O.pi_factor(2.0, 0.25) - 0.8 * 2.0 ** -0.175 * 0.25 ** 0.1) < 1e-15
    assert O.pi_factor(1e-30, 1.0) == 2.5 and O.pi_factor(1e9, 1.0) == 0.3 and O.pi_factor(float("nan"), 1.0) == 0.3


def test_adaptive_controller_on_a_scalar_ode():
    """u' = -u + sin(10 t) from 0 to 2: reaches t1 exactly, a too-large first step is rejected, accepted errors are <= 1,
    step factors stay inside the clip, and the global error follows the tolerance."""
    def run(tol, dt0):
        tt = [0.0]     # the controller does not pass t: carry it as a state component (t' = 1)
        f = lambda us: [np.array([-us[0][0] + np.sin(10 * us[0][1]), 1.0])]
        u, hist = O.rk45_adaptive(f, [np.array([1.0, 0.0])], 0.0, 2.0, dt0, tol, tol)
        return u[0], hist
    exact = lambda t: (1 + 10 / 101) * np.exp(-t) + (np.sin(10 * t) - 10 * np.cos(10 * t)) / 101
    errs = []
    for tol in (1e-5, 1e-7, 1e-9):
        u, hist = run(tol, 1.0)
        assert abs(u[1] - 2.0) < 1e-14                       # t reached exactly (t' = 1 is integrated exactly)
        assert abs(sum(h[0] for h in hist if h[2]) - 2.0) < 1e-12
        assert not hist[0][2] and hist[0][0] == 1.0           # dt0 = 1 is far too large
        assert all(h[1] <= 1.0 for h in hist if h[2]) and all(h[1] > 1.0 for h in hist if not h[2])
        for (d0, e0, _), (d1, _, _) in zip(hist[:-2], hist[1:-1]):
            assert 0.3 - 1e-12 <= d1 / d0 <= 2.5 + 1e-12
        errs.append(abs(u[0] - exact(2.0)))
        assert errs[-1] < 50 * tol
    assert errs[0] > errs[1] > errs[2]
    assert sum(1 for h in run(1e-9, 1.0)[1] if h[2]) > 2 * sum(1 for h in run(1e-5, 1.0)[1] if h[2])
