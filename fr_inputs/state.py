"""Seeded synthetic initial states (conserved variables rho, rho*v, E on the physical solution points).

Only input data: closed-form fields and seeded perturbations.  All random
draws use numpy.random.Generator(PCG64(seed)), drawn once in canonical order (type, solution point,
variable, element).  States are arrays [N_u, 5, N_e] per element type.
"""
import numpy as np

GAMMA = 1.4


def prim_to_cons(rho, v, p, gamma=GAMMA):
    """rho [...], v [3,...], p [...] -> u [5,...]."""
    E = p / (gamma - 1) + 0.5 * rho * (v[0] ** 2 + v[1] ** 2 + v[2] ** 2)
    return np.stack([rho, rho * v[0], rho * v[1], rho * v[2], E], axis=0)


def freestream(xu, rho=1.0, v=(0.3, 0.0, 0.0), p=1.0 / GAMMA, gamma=GAMMA):
    """Uniform state on points xu [N_u, N_e, 3] -> [N_u, 5, N_e]."""
    nu, ne, _ = xu.shape
    u = prim_to_cons(np.float64(rho), np.array(v, dtype=np.float64), np.float64(p), gamma)
    return np.broadcast_to(u[None, :, None], (nu, 5, ne)).copy()


def perturb(us, amp, seed, rho=1.0, v=(0.3, 0.0, 0.0), p=1.0 / GAMMA, gamma=GAMMA):
    """u_k <- u_k + amp * s_k * U(-1,1), s = (rho, rho|v|, rho|v|, rho|v|, E)  (reading R17). `us`: list per type."""
    rng = np.random.Generator(np.random.PCG64(seed))
    vm = float(np.sqrt(sum(c * c for c in v)))
    E = p / (gamma - 1) + 0.5 * rho * vm * vm
    s = np.array([rho, rho * vm, rho * vm, rho * vm, E])
    return [u + amp * s[None, :, None] * rng.uniform(-1.0, 1.0, size=u.shape) for u in us]


def isentropic_vortex(xu, gamma=GAMMA, eps=5.0, R=0.1, centre=(0.5, 0.5), vinf=(1.0, 1.0, 0.0), length=1.0, t=0.0):
    """Config-2 state (reading R20): z-invariant isentropic vortex, rho_inf = p_inf = 1.
    The nearest periodic image of the (advected) centre is used so the field is periodic to ~e^-12."""
    x0 = (centre[0] + vinf[0] * t) % length
    y0 = (centre[1] + vinf[1] * t) % length
    dx = xu[..., 0] - x0
    dy = xu[..., 1] - y0
    dx -= length * np.round(dx / length)
    dy -= length * np.round(dy / length)
    r2 = (dx * dx + dy * dy) / (R * R)
    f = eps / (2 * np.pi) * np.exp(0.5 * (1 - r2))
    vx = vinf[0] - f * dy / R
    vy = vinf[1] + f * dx / R
    vz = np.full_like(vx, vinf[2])
    T = 1 - (gamma - 1) * eps * eps / (8 * gamma * np.pi ** 2) * np.exp(1 - r2)
    rho = T ** (1 / (gamma - 1))
    p = rho * T
    return np.ascontiguousarray(prim_to_cons(rho, np.stack([vx, vy, vz]), p, gamma).transpose(1, 0, 2))


def smooth_periodic(xu, length=1.0, gamma=GAMMA):
    """Smooth periodic manufactured field for consistency-order tests.
    Returns the state and the primitive fields' closed forms are in tests (sympy)."""
    k = 2 * np.pi / length
    x, y, z = xu[..., 0], xu[..., 1], xu[..., 2]
    rho = 1 + 0.2 * np.sin(k * (x + y + z))
    vx = 0.5 + 0.1 * np.cos(k * (x - 2 * y))
    vy = 0.3 + 0.1 * np.sin(k * (y + z))
    vz = 0.2 + 0.1 * np.cos(k * (z - x))
    p = 1 + 0.1 * np.cos(k * (x + y - z))
    return np.ascontiguousarray(prim_to_cons(rho, np.stack([vx, vy, vz]), p, gamma).transpose(1, 0, 2))
