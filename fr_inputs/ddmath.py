"""Double-double (~32 significant digits) dense linear algebra on numpy arrays.

Used only by `fr_inputs.refelem` to invert the (ill-conditioned) monomial
Vandermonde / Gram matrices of the reference elements so that the operator
matrices handed to `fr_setup` and to the oracle are correctly rounded FP64.
A number is a pair (hi, lo) of float64 arrays with |lo| <= ulp(hi)/2.
Nothing here knows about flux reconstruction.
"""
import numpy as np

_SPLIT = 134217729.0  # 2**27 + 1 (Veltkamp)


def _two_sum(a, b):
    s = a + b
    bb = s - a
    return s, (a - (s - bb)) + (b - bb)


def _quick_two_sum(a, b):
    s = a + b
    return s, b - (s - a)


def _split(a):
    t = _SPLIT * a
    hi = t - (t - a)
    return hi, a - hi


def _two_prod(a, b):
    p = a * b
    ah, al = _split(a)
    bh, bl = _split(b)
    return p, ((ah * bh - p) + ah * bl + al * bh) + al * bl


class DD:
    """Array of double-double numbers."""
    __slots__ = ("hi", "lo")

    def __init__(self, hi, lo=None):
        self.hi = np.array(hi, dtype=np.float64)
        self.lo = np.zeros_like(self.hi) if lo is None else np.array(lo, dtype=np.float64)

    # ---- construction / conversion
    @staticmethod
    def from_mp(arr):
        """From a (nested) sequence / object array of mpmath numbers."""
        a = np.asarray(arr, dtype=object)
        hi = np.vectorize(float, otypes=[np.float64])(a)
        lo = np.vectorize(lambda x, h: float(x - h), otypes=[np.float64])(a, hi)
        return DD(hi, lo)

    def to_f64(self):
        return self.hi + self.lo

    @property
    def shape(self):
        return self.hi.shape

    def __getitem__(self, k):
        return DD(self.hi[k], self.lo[k])

    def __setitem__(self, k, v):
        self.hi[k] = v.hi
        self.lo[k] = v.lo

    def copy(self):
        return DD(self.hi.copy(), self.lo.copy())

    @property
    def T(self):
        return DD(self.hi.T, self.lo.T)

    def reshape(self, *s):
        return DD(self.hi.reshape(*s), self.lo.reshape(*s))

    # ---- arithmetic
    def __neg__(self):
        return DD(-self.hi, -self.lo)

    def __add__(self, o):
        o = _as_dd(o)
        s1, s2 = _two_sum(self.hi, o.hi)
        t1, t2 = _two_sum(self.lo, o.lo)
        s2 = s2 + t1
        s1, s2 = _quick_two_sum(s1, s2)
        s2 = s2 + t2
        s1, s2 = _quick_two_sum(s1, s2)
        return DD(s1, s2)

    __radd__ = __add__

    def __sub__(self, o):
        return self + (-_as_dd(o))

    def __rsub__(self, o):
        return _as_dd(o) + (-self)

    def __mul__(self, o):
        o = _as_dd(o)
        p, e = _two_prod(self.hi, o.hi)
        e = e + (self.hi * o.lo + self.lo * o.hi)
        p, e = _quick_two_sum(p, e)
        return DD(p, e)

    __rmul__ = __mul__

    def __truediv__(self, o):
        o = _as_dd(o)
        q1 = self.hi / o.hi
        r = self - o * q1
        q2 = r.hi / o.hi
        r = r - o * q2
        q3 = r.hi / o.hi
        s, e = _quick_two_sum(q1, q2)
        return DD(s, e) + DD(q3)


def _as_dd(x):
    return x if isinstance(x, DD) else DD(np.asarray(x, dtype=np.float64))


def dd_zeros(shape):
    return DD(np.zeros(shape))


def dd_eye(n):
    return DD(np.eye(n))


def dd_matmul(a, b):
    """(M,K) @ (K,N) accumulated in double-double, k ascending."""
    m, k = a.shape
    k2, n = b.shape
    assert k == k2
    acc = dd_zeros((m, n))
    for kk in range(k):
        acc = acc + DD(a.hi[:, kk:kk + 1], a.lo[:, kk:kk + 1]) * DD(b.hi[kk:kk + 1, :], b.lo[kk:kk + 1, :])
    return acc


def dd_inv(a):
    """Gauss-Jordan inverse with partial pivoting, all in double-double."""
    n = a.shape[0]
    assert a.shape == (n, n)
    aug = DD(np.concatenate([a.hi, np.eye(n)], axis=1), np.concatenate([a.lo, np.zeros((n, n))], axis=1))
    for k in range(n):
        piv = k + int(np.argmax(np.abs(aug.hi[k:, k])))
        if aug.hi[piv, k] == 0.0:
            raise np.linalg.LinAlgError("singular matrix in dd_inv")
        if piv != k:
            aug.hi[[k, piv]] = aug.hi[[piv, k]]
            aug.lo[[k, piv]] = aug.lo[[piv, k]]
        row = aug[k] / aug[k, k]
        aug[k] = row
        f = DD(aug.hi[:, k:k + 1].copy(), aug.lo[:, k:k + 1].copy())
        f.hi[k] = 0.0
        f.lo[k] = 0.0
        upd = f * DD(row.hi[None, :], row.lo[None, :])
        aug = aug - upd
    return DD(aug.hi[:, n:], aug.lo[:, n:])


def dd_pow(x, e):
    """x**e for a non-negative integer array/scalar exponent e (elementwise, by repeated multiply)."""
    e = np.broadcast_to(np.asarray(e, dtype=np.int64), x.shape)
    out = DD(np.ones(x.shape))
    for k in range(int(e.max()) if e.size else 0):
        mask = e > k
        nxt = out * x
        out = DD(np.where(mask, nxt.hi, out.hi), np.where(mask, nxt.lo, out.lo))
    return out
