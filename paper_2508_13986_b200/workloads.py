"""Seeded synthetic inputs for BASELINE.json's configs (shared by tests, bench and the oracle
harness). Holds none of the method's arithmetic: only parameters, initial conditions and the
measurement values z (drawn around a truth trajectory integrated with classic RK4)."""
import numpy as np

S0 = 250813986  # base seed

DYN_L63, DYN_L63_PAPER, DYN_L96, DYN_LINEAR, DYN_CONST = 0, 1, 2, 3, 4


def lorenz63(x, s=10.0, b=8.0 / 3.0, r=28.0):
    return np.array([s * (x[1] - x[0]), x[0] * (r - x[2]) - x[1], x[0] * x[1] - b * x[2]])


def rk4_truth(f, x0, t_end, h=1e-3):
    x = np.array(x0, dtype=np.float64)
    for _ in range(int(round(t_end / h))):
        k1 = f(x); k2 = f(x + 0.5 * h * k1); k3 = f(x + 0.5 * h * k2); k4 = f(x + h * k3)
        x = x + h / 6.0 * (k1 + 2 * k2 + 2 * k3 + k4)
    return x


def config0():
    """Lorenz '63 3-D, smallest instance: 20 steps, prune every step."""
    return dict(name="cfg0_lorenz63_small", n=3, dyn=DYN_L63, params=[10.0, 8.0 / 3.0, 28.0], dx=[0.5] * 3,
                thresh=2e-5, cfl=0.9, mean=[-11.5, -10.0, 9.5], cov=np.eye(3), steps=20, prune_every=1,
                max_cells=1 << 16)


def config1():
    """Lorenz '63 3-D full run to t=1 with Bayesian corrections at t=0.5 and t=1.0 (R = I)."""
    c = config0()
    w = np.random.default_rng(S0 + 1).standard_normal((2, 3))
    mean = np.array(c["mean"])
    z1 = rk4_truth(lorenz63, mean, 0.5) + w[0]
    z2 = rk4_truth(lorenz63, mean, 1.0) + w[1]
    c.update(name="cfg1_lorenz63_full", dx=[0.3] * 3, t_meas=[0.5, 1.0], z=[z1, z2], R=np.eye(3), steps=None,
             max_cells=1 << 21)
    return c


def config2():
    """Lorenz '96 6-D (headline): propagate to t=0.5, prune every 5 steps."""
    return dict(name="cfg2_lorenz96_6d", n=6, dyn=DYN_L96, params=[4.0], dx=[0.5] * 6, thresh=1e-7, cfl=0.9,
                mean=[4.01, 4.0, 4.0, 4.0, 4.0, 4.0], cov=0.25 * np.eye(6), t_end=0.5, prune_every=5,
                max_cells=1 << 25)


def config3(dx=0.35):
    """Synthetic 6-D stress: linear rotation-plus-shear f = A x, spectral radius <= 1, 50 steps."""
    A = np.random.default_rng(S0 + 3).normal(0.0, 0.3, (6, 6))
    rho = np.max(np.abs(np.linalg.eigvals(A)))
    if rho > 1.0:
        A = A / rho
    return dict(name="cfg3_linear_6d", n=6, dyn=DYN_LINEAR, params=A.ravel(), dx=[dx] * 6, thresh=1e-10, cfl=0.9,
                mean=[0.0] * 6, cov=np.eye(6), steps=50, prune_every=5, max_cells=3 << 25)


def config4_keys(K, seed=S0 + 4):
    """Hashtable microbench keys: 6-D coords uniform in [-512, 511], 10 bits each, distinct."""
    rng = np.random.default_rng(seed)
    c = rng.integers(-512, 512, (int(1.01 * K) + 16, 6))
    k = np.zeros(len(c), dtype=np.uint64)
    for j in range(6):
        k |= (c[:, j] + 512).astype(np.uint64) << np.uint64(10 * (5 - j))
    _, first = np.unique(k, return_index=True)
    return k[np.sort(first)][:K]
