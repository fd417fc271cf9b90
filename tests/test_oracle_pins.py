"""Pins for the CPU oracle: the oracle is checked against closed forms,
invariants, textbook special cases and an independent dense-array implementation -- never
against itself and never against the CUDA path."""
import itertools
import math

import numpy as np
import pytest

from oracle import dense_ctu
from oracle.binding import Oracle

S0 = 250813986


def box(lo, hi):
    """All integer coordinates c with lo <= c < hi (lexicographic)."""
    return np.array(list(itertools.product(*[range(a, b) for a, b in zip(lo, hi)])), dtype=np.int32)


def raw(n, h, dyn, params, keys, p, origin=None, cfl=0.9, hi_res=1, limiter=0, grow=False):
    o = Oracle(n, h, 1e-300, dyn, params, cfl=cfl, hi_res=hi_res, limiter=limiter)
    o.set_flags(grow=grow, normalise=False)
    o.import_state(np.zeros(n) if origin is None else origin, keys, p)
    return o


def as_dict(keys, p):
    return {tuple(k): v for k, v in zip(keys.tolist(), p.tolist())}


# ---- P1 telescoping / conservation -------------------------------------------------------------
@pytest.mark.parametrize("n,dyn,params", [(3, 0, [10, 8 / 3, 28]), (4, 2, [4.0]), (6, 2, [4.0])])
def test_P1_conservation_when_support_is_two_cells_inside(n, dyn, params):
    rng = np.random.default_rng(S0 + 101 + n)
    side = {3: 9, 4: 7, 6: 5}[n]
    keys = box([0] * n, [side] * n)
    inner = np.all((keys >= 2) & (keys < side - 2), axis=1)
    p = np.where(inner, rng.random(len(keys)), 0.0)
    for ragged in (False, True):
        k2, p2 = keys, p
        if ragged:
            # ragged active set: with d = sum_j (distance of coordinate j outside the support's box), a random
            # 30 % of the zero cells with d >= 3 are dropped. Cells that then miss a face neighbour have
            # d >= 2, so they and all their face neighbours (d >= 1) carry no mass: P1's premise holds.
            d = np.sum(np.maximum(2 - keys, 0) + np.maximum(keys - (side - 3), 0), axis=1)
            drop = (d >= 3) & (rng.random(len(keys)) < 0.3)
            assert drop.sum() > 0
            k2, p2 = keys[~drop], p2[~drop]
        o = raw(n, [0.5] * n, dyn, params, k2, p2, origin=[1.0] * n)
        o.step()
        _, p1 = o.export()
        assert len(p1) == len(p2)
        assert abs(p1.sum() - p2.sum()) <= len(k2) * 2.0 ** -52 * p2.sum()
        assert abs(o.last_mass() - p2.sum()) <= len(k2) * 2.0 ** -52 * p2.sum()


def test_P1_mass_is_lost_only_through_boundary_faces():
    # 1-D, u>0 everywhere, all cells carry mass: the only loss is the outflow of the last cell.
    n, h, v = 1, [0.5], [1.0]
    keys = box([0], [8])
    p = np.arange(1, 9, dtype=np.float64)
    o = raw(n, h, 4, v, keys, p, hi_res=0, cfl=0.5)
    dt = o.step()
    assert dt == 0.5 / (1.0 / 0.5)
    _, p1 = o.export()
    assert p1.sum() == pytest.approx(p.sum() - dt / 0.5 * 1.0 * p[-1], rel=1e-15)


# ---- P2 Courant-1 shift, bit exact ----------------------------------------------------------------
@pytest.mark.parametrize("n,axis,sign", [(1, 0, 1), (1, 0, -1), (3, 1, 1), (3, 2, -1), (6, 4, 1), (6, 0, -1)])
def test_P2_courant_one_shift_is_bit_exact(n, axis, sign):
    rng = np.random.default_rng(S0 + 102)
    v = np.zeros(n)
    v[axis] = 2.0 * sign
    lo, hi = [0] * n, [3] * n
    hi[axis] = 12
    keys = box(lo, hi)
    p = rng.integers(0, 64, len(keys)).astype(np.float64) * 2.0 ** -9
    edge = (keys[:, axis] < 2) | (keys[:, axis] >= 10)
    p[edge] = 0.0
    for hi_res, limiter in [(0, 0), (1, 0), (1, 1)]:
        o = raw(n, [0.5] * n, 4, v, keys, p, cfl=1.0, hi_res=hi_res, limiter=limiter)
        dt = o.step()
        assert dt == 0.25
        k1, p1 = o.export()
        d0, d1 = as_dict(keys, p), as_dict(k1, p1)
        for k, val in d1.items():
            src = list(k)
            src[axis] -= sign
            assert val == d0.get(tuple(src), 0.0)  # bit exact


# ---- P3 n-D constant-velocity closed form, all 2^n sign patterns ---------------------------------
def closed_form_ctu(P, nu, sgn):
    """P' = P - sum_j nu_j D_j P + sum_{j<l} nu_j nu_l D_j D_l P, D_j = upwind difference."""
    n = P.ndim

    def D(A, j):
        return A - np.roll(A, sgn[j], axis=j)

    out = P.copy()
    for j in range(n):
        out = out - nu[j] * D(P, j)
    for j in range(n):
        for l in range(j + 1, n):
            out = out + nu[j] * nu[l] * D(D(P, j), l)
    return out


@pytest.mark.parametrize("n,side", [(2, 9), (3, 7), (6, 5)])
def test_P3_constant_velocity_closed_form_all_sign_patterns(n, side):
    rng = np.random.default_rng(S0 + 103 + n)
    h = np.array([0.5, 0.25, 1.0, 0.5, 2.0, 0.75][:n])
    keys = box([0] * n, [side] * n)
    Pd = np.zeros([side] * n)
    inner = tuple([slice(2, side - 2)] * n)
    Pd[inner] = rng.random(Pd[inner].shape)
    p = Pd[tuple(keys.T)]
    for sgn in itertools.product([1, -1], repeat=n):
        speed = rng.uniform(0.3, 1.5, n)
        v = speed * np.array(sgn)
        o = raw(n, h, 4, v, keys, p, cfl=0.9, hi_res=0)
        dt = o.step()
        nu = speed * dt / h
        assert nu.sum() == pytest.approx(0.9, rel=1e-14)
        k1, p1 = o.export()
        got = np.zeros_like(Pd)
        got[tuple(k1.T)] = p1
        want = closed_form_ctu(Pd, nu, sgn)
        sl = tuple([slice(1, side - 1)] * n)
        assert np.max(np.abs(got[sl] - want[sl])) <= 1e-14 * np.max(np.abs(want))


# ---- P4 1-D DCU binomial smear ------------------------------------------------------------------------
def test_P4_dcu_binomial_smear():
    N, k, nu = 64, 10, 0.4
    keys = box([0], [N])
    p = np.where((keys[:, 0] >= 10) & (keys[:, 0] < 20), 1.0, 0.0)
    o = raw(1, [0.5], 4, [1.0], keys, p, hi_res=0, cfl=1.0)
    for _ in range(k):
        assert o.step(nu * 0.5) == nu * 0.5
    _, p1 = o.export()
    want = np.zeros(N)
    for m in range(k + 1):
        w = math.comb(k, m) * nu ** m * (1 - nu) ** (k - m)
        want[m:] += w * p[: N - m]
    assert np.max(np.abs(p1 - want)) < 1e-13


# ---- P5 Lax-Wendroff with phi == 1 ---------------------------------------------------------------------
@pytest.mark.parametrize("sign", [1, -1])
def test_P5_unlimited_hires_is_lax_wendroff(sign):
    rng = np.random.default_rng(S0 + 105)
    N, nu = 40, 0.37
    keys = box([0], [N])
    p = np.zeros(N)
    p[5:35] = rng.random(30)
    o = raw(1, [0.25], 4, [2.0 * sign], keys, p, hi_res=1, limiter=1, cfl=1.0)
    dt = nu * 0.25 / 2.0
    assert o.step(dt) == dt
    _, p1 = o.export()
    c = nu * sign
    want = p - c / 2 * (np.roll(p, -1) - np.roll(p, 1)) + c * c / 2 * (np.roll(p, -1) - 2 * p + np.roll(p, 1))
    assert np.max(np.abs(p1[2:-2] - want[2:-2])) < 1e-14


# ---- P6 MC limiter: TVD and order of accuracy --------------------------------------------------------
def test_P6_mc_limiter_is_tvd_on_step_data():
    N = 80
    keys = box([0], [N])
    p = np.where((keys[:, 0] >= 10) & (keys[:, 0] < 30), 1.0, 0.0)
    o = raw(1, [0.5], 4, [1.0], keys, p, hi_res=1, limiter=0, cfl=0.8)
    tv = np.abs(np.diff(p)).sum()
    for _ in range(40):
        o.step()
        _, p1 = o.export()
        tv1 = np.abs(np.diff(p1)).sum()
        assert tv1 <= tv * (1 + 1e-14)
        tv = tv1
        assert p1.min() >= -1e-15 and p1.max() <= 1 + 1e-14


def _advect_gaussian_error(N, hi_res):
    h, v, nu, L = 1.0 / N, 1.0, 0.8, 1.0
    keys = box([-2 * N], [4 * N])
    x = keys[:, 0] * h
    f = lambda y: np.exp(-0.5 * ((y - 0.5) / 0.08) ** 2)
    o = raw(1, [h], 4, [v], keys, f(x), hi_res=hi_res, cfl=1.0)
    steps = int(round(L / (nu * h)))
    for _ in range(steps):
        o.step(nu * h / v)
    _, p1 = o.export()
    return h * np.abs(p1 - f(x - v * o.time())).sum()


def test_P6_second_order_with_hires_first_order_without():
    e1, e2 = _advect_gaussian_error(100, 1), _advect_gaussian_error(200, 1)
    assert 1.7 <= math.log2(e1 / e2) <= 2.3
    f1, f2 = _advect_gaussian_error(100, 0), _advect_gaussian_error(200, 0)
    assert 0.6 <= math.log2(f1 / f2) <= 1.2
    assert e2 < f2 / 10


# ---- P7 brute force: dense gather form vs sparse scatter form ---------------------------------------
CASES_P7 = [
    (3, 6, 0, [10, 8 / 3, 28], [-11.5, -10, 9.5]),
    (3, 6, 1, [4.0, 1.0, 48.0], [-11.5, -10, 9.5]),
    (4, 4, 2, [4.0], [4.01, 4, 4, 4]),
    (6, 3, 2, [4.0], [4.01, 4, 4, 4, 4, 4]),
    (6, 3, 3, None, [0.3, -0.2, 0.1, 0.5, -0.4, 0.2]),
]


@pytest.mark.parametrize("n,side,dyn,params,origin", CASES_P7)
@pytest.mark.parametrize("ragged", [False, True])
def test_P7_dense_gather_form_equals_sparse_scatter_form(n, side, dyn, params, origin, ragged):
    rng = np.random.default_rng(S0 + 107 + 10 * n + dyn + ragged)
    if params is None:
        params = rng.normal(0, 0.3, (n, n)).ravel()
    h = rng.uniform(0.3, 0.6, n)
    keys = box([-(side // 2)] * n, [side - side // 2] * n)
    if ragged:
        keys = keys[rng.random(len(keys)) < 0.6]
    p = rng.random(len(keys)) - 0.1  # a few negatives: no clipping anywhere (A5)
    order = np.lexsort(keys.T[::-1])
    keys, p = keys[order], p[order]
    for hi_res, limiter in [(0, 0), (1, 0), (1, 1)]:
        o = raw(n, h, dyn, params, keys, p, origin=origin, hi_res=hi_res, limiter=limiter)
        dt = o.step()
        k1, p1 = o.export()
        assert np.array_equal(k1, keys)
        want = dense_ctu.dense_step_sparse(keys, p, dyn, params, origin, h, dt, bool(hi_res), limiter)
        assert np.max(np.abs(p1 - want)) <= 1e-13 * np.max(np.abs(want))


# ---- P8 dt closed forms (Eq. 8) --------------------------------------------------------------------------
def test_P8_dt_constant_velocity_exact():
    v, h = [1.5, -0.25, 3.0], [0.5, 0.125, 2.0]
    o = raw(3, h, 4, v, box([0] * 3, [3] * 3), np.ones(27), cfl=0.9)
    assert o.step() == 0.9 / (1.5 / 0.5 + 0.25 / 0.125 + 3.0 / 2.0)
    assert o.step(1e-3) == 1e-3  # caller's cap binds
    assert o.step(float("inf")) == 0.9 / 6.5 and o.step(-1.0) == 0.9 / 6.5


def test_P8_dt_linear_dynamics_brute_force():
    rng = np.random.default_rng(S0 + 108)
    n, A = 3, rng.normal(0, 0.3, (3, 3))
    h, origin = np.array([0.5, 0.4, 0.3]), np.array([0.2, -0.1, 0.3])
    keys = box([-4, -3, -5], [5, 4, 3])
    o = raw(n, h, 3, A.ravel(), keys, np.ones(len(keys)), origin=origin, cfl=0.9)
    s = np.zeros(len(keys))
    for j in range(n):
        xf = origin + keys * h
        xf[:, j] -= 0.5 * h[j]
        s += np.abs(xf @ A[j]) / h[j]
    assert o.step() == pytest.approx(0.9 / s.max(), rel=1e-15)


def test_A12_face_velocity_matches_independent_numpy():
    rng = np.random.default_rng(S0 + 112)
    for n, dyn, params in [(3, 0, [10, 8 / 3, 28]), (3, 1, [4, 1, 48]), (6, 2, [4.0]), (4, 2, [8.0]),
                           (5, 3, rng.normal(0, 0.3, 25))]:
        h, origin = rng.uniform(0.2, 0.6, n), rng.normal(0, 3, n)
        o = raw(n, h, dyn, params, np.zeros((1, n), dtype=np.int32), [1.0], origin=origin)
        for _ in range(20):
            c = rng.integers(-30, 30, n).astype(np.int32)
            for j in range(n):
                x = [np.float64(origin[m] + (c[m] - (0.5 if m == j else 0.0)) * h[m]) for m in range(n)]
                want = float(dense_ctu.dynamics(dyn, params, x, j))
                assert o.face_velocity(c, j) == pytest.approx(want, rel=1e-13, abs=1e-13)


# ---- dynamics pins: what the paper and the mathematics fix about f(x), with no second typing of f ------
def _oracle_for(n, dyn, params):
    return raw(n, [0.5] * n, dyn, params, np.zeros((1, n), dtype=np.int32), [1.0])


def _jacobian(o, x, eps=0.5):
    """Central differences; exact up to rounding for the (at most quadratic) Lorenz fields."""
    n = len(x)
    J = np.zeros((n, n))
    for m in range(n):
        e = np.zeros(n); e[m] = eps
        J[:, m] = (o.dynamics(x + e) - o.dynamics(x - e)) / (2 * eps)
    return J


@pytest.mark.parametrize("n", [4, 5, 6])
def test_D_lorenz96_equilibrium_energy_divergence(n):
    # f_j = (x_{j+1} - x_{j-2}) x_{j-1} - x_j + F, cyclic; "(F, ..., F) is an unstable equilibrium"
    F = 4.0
    o = _oracle_for(n, 2, [F])
    assert np.array_equal(o.dynamics(np.full(n, F)), np.zeros(n))          # exactly: (F - F) F - F + F
    rng = np.random.default_rng(S0 + 300 + n)
    for _ in range(20):
        x = rng.normal(0, 3, n)
        f = o.dynamics(x)
        # the quadratic (advection) term conserves energy: sum_j x_j (x_{j+1} - x_{j-2}) x_{j-1} = 0.
        # Any wrong cyclic index (x_{j+2} for x_{j-2}, x_{j+1} for x_{j-1}, ...) breaks the cancellation.
        quad = f + x - F
        assert abs(np.dot(x, quad)) <= 1e-12 * np.sum(np.abs(x) ** 3 + 1)
        J = _jacobian(o, x)
        assert np.allclose(np.diag(J), -1.0, atol=1e-12)                   # div f = -n
        # Jacobian structure of the printed formula: df_j/dx_{j+1} = x_{j-1}, df_j/dx_{j-2} = -x_{j-1},
        # df_j/dx_{j-1} = x_{j+1} - x_{j-2}; everything else 0
        for j in range(n):
            want = np.zeros(n)
            want[j] += -1.0
            want[(j + 1) % n] += x[(j - 1) % n]
            want[(j - 2) % n] += -x[(j - 1) % n]
            want[(j - 1) % n] += x[(j + 1) % n] - x[(j - 2) % n]
            assert np.allclose(J[j], want, atol=1e-11), (j, J[j], want)
    # instability of (F,...,F): the Jacobian there has an eigenvalue with positive real part (n = 6, F = 4)
    if n == 6:
        assert np.max(np.linalg.eigvals(_jacobian(o, np.full(n, F))).real) > 0.1


def test_D_lorenz63_classic_fixed_points_divergence_symmetry():
    # BASELINE.json configs[0-1]: classic Lorenz '63, (sigma, beta, rho) = (10, 8/3, 28)
    s_, b_, r_ = 10.0, 8.0 / 3.0, 28.0
    o = _oracle_for(3, 0, [s_, b_, r_])
    q = math.sqrt(b_ * (r_ - 1.0))
    assert np.array_equal(o.dynamics(np.zeros(3)), np.zeros(3))
    for sgn in (1.0, -1.0):
        assert np.allclose(o.dynamics(np.array([sgn * q, sgn * q, r_ - 1.0])), 0.0, atol=1e-12)
    rng = np.random.default_rng(S0 + 310)
    for _ in range(10):
        x = rng.normal(0, 10, 3)
        J = _jacobian(o, x)
        assert np.trace(J) == pytest.approx(-(s_ + 1.0 + b_), abs=1e-10)    # div f = -(sigma + 1 + beta)
        want = np.array([[-s_, s_, 0.0], [r_ - x[2], -1.0, -x[0]], [x[1], x[0], -b_]])
        assert np.allclose(J, want, atol=1e-9)
        # symmetry (x1, x2, x3) -> (-x1, -x2, x3)
        f, g = o.dynamics(x), o.dynamics(x * np.array([-1.0, -1.0, 1.0]))
        assert np.allclose(g, f * np.array([-1.0, -1.0, 1.0]), atol=1e-12)


def test_D_lorenz63_paper_form_fixed_points_divergence():
    # f = (sigma (x2 - x1), -x2 - x1 x3, -b x3 + x1 x2 - b r), (sigma, b, r) = (4, 1, 48)
    s_, b_, r_ = 4.0, 1.0, 48.0
    o = _oracle_for(3, 1, [s_, b_, r_])
    # fixed points: x1 = x2; x2 (1 + x3) = 0 -> (0, 0, -r) and x3 = -1, x1^2 = b (r - 1)
    assert np.allclose(o.dynamics(np.array([0.0, 0.0, -r_])), 0.0, atol=1e-13)
    q = math.sqrt(b_ * (r_ - 1.0))
    for sgn in (1.0, -1.0):
        assert np.allclose(o.dynamics(np.array([sgn * q, sgn * q, -1.0])), 0.0, atol=1e-12)
    assert np.allclose(o.dynamics(np.zeros(3)), [0.0, 0.0, -b_ * r_])
    rng = np.random.default_rng(S0 + 311)
    for _ in range(10):
        x = rng.normal(0, 10, 3)
        J = _jacobian(o, x)
        assert np.trace(J) == pytest.approx(-(s_ + 1.0 + b_), abs=1e-10)
        want = np.array([[-s_, s_, 0.0], [-x[2], -1.0, -x[0]], [x[1], x[0], -b_]])
        assert np.allclose(J, want, atol=1e-9)
    # it is the classic system with z shifted by r: f_paper(x1, x2, x3) = f_classic(x1, x2, x3 + r)
    oc = _oracle_for(3, 0, [s_, b_, r_])
    x = rng.normal(0, 5, 3)
    assert np.allclose(o.dynamics(x), oc.dynamics(x + np.array([0.0, 0.0, r_])), atol=1e-10)


def test_D_linear_and_constant_dynamics_are_what_they_say():
    rng = np.random.default_rng(S0 + 312)
    A = rng.normal(0, 0.3, (5, 5))
    o = _oracle_for(5, 3, A.ravel())
    x = rng.normal(0, 2, 5)
    assert np.allclose(_jacobian(o, x), A, atol=1e-12)                      # f = A x: Jacobian is A (row-major)
    assert np.array_equal(o.dynamics(np.zeros(5)), np.zeros(5))
    v = rng.normal(0, 1, 4)
    oc = _oracle_for(4, 4, v)
    assert np.array_equal(oc.dynamics(rng.normal(0, 1, 4)), v)


def test_D_face_velocity_is_the_dynamics_at_the_lower_face_centre():
    # Eq. (7) text: the flux velocity is f_j at the centre of face i - e^j / 2
    rng = np.random.default_rng(S0 + 313)
    n, h, origin = 6, rng.uniform(0.2, 0.6, 6), rng.normal(0, 3, 6)
    o = raw(n, h, 2, [4.0], np.zeros((1, n), dtype=np.int32), [1.0], origin=origin)
    for _ in range(10):
        c = rng.integers(-30, 30, n).astype(np.int32)
        for j in range(n):
            x = origin + c * h
            x[j] = origin[j] + (c[j] - 0.5) * h[j]
            assert o.face_velocity(c, j) == o.dynamics(x)[j]


# ---- P9 linear dynamics: grid moments follow N(e^{At} mu, e^{At} Sigma e^{A^T t}) ---------------------
def _moments(keys, p, origin, h):
    x = origin + keys * h
    m = (p[:, None] * x).sum(0)
    d = x - m
    return m, (p[:, None, None] * d[:, :, None] * d[:, None, :]).sum(0)


def _expm(A, t):
    w, V = np.linalg.eig(A)
    return (V @ np.diag(np.exp(w * t)) @ np.linalg.inv(V)).real


def test_P9_linear_dynamics_moments_full_pipeline():
    A = np.array([[-0.1, 1.0], [-1.0, -0.2]])
    mu0, cov0, T = np.array([2.0, 0.5]), np.array([[0.09, 0.02], [0.02, 0.05]]), 0.8
    errs = []
    for dx in (0.06, 0.03):
        o = Oracle(2, [dx, dx], 1e-9, 3, A.ravel(), cfl=0.9)
        o.init_gaussian(mu0, cov0)
        k = 0
        while o.time() < T:
            o.step(T - o.time())
            k += 1
            if k % 3 == 0:
                o.prune()
        keys, p = o.export()
        assert p.sum() == pytest.approx(1.0, abs=1e-12)
        m, S = _moments(keys, p, mu0, np.array([dx, dx]))
        E = _expm(A, T)
        errs.append((np.abs(m - E @ mu0).max(), np.abs(S - E @ cov0 @ E.T).max() / np.abs(cov0).max()))
    assert errs[1][0] < 2e-3 and errs[1][1] < 0.02      # discretisation-limited
    assert errs[1][1] < errs[0][1] / 2.5                # improves ~4x per halving (2nd order)


# ---- P10 correction: direct Bayes product and Kalman moments -----------------------------------------------
def test_P10_correction_direct_and_kalman():
    n, dx = 3, 0.2
    mu0, cov0 = np.array([-11.5, -10, 9.5]), np.diag([1.0, 0.5, 0.8])
    z, R = np.array([-11.0, -10.4, 9.9]), np.array([[1.0, 0.2, 0], [0.2, 0.7, 0.1], [0, 0.1, 1.2]])
    o = Oracle(n, [dx] * n, 1e-9, 0, [10, 8 / 3, 28])
    o.init_gaussian(mu0, cov0)
    keys, p0 = o.export()
    o.correct(z, R)
    k1, p1 = o.export()
    assert np.array_equal(keys, k1)
    d = z - (mu0 + keys * dx)
    L = np.exp(-0.5 * np.einsum("ij,jk,ik->i", d, np.linalg.inv(R), d))
    want = p0 * L / (p0 * L).sum()
    assert np.max(np.abs(p1 - want)) <= 1e-13 * want.max()  # summation order over 47k cells
    K = cov0 @ np.linalg.inv(cov0 + R)
    m, S = _moments(keys, p1, mu0, np.array([dx] * n))
    assert np.abs(m - (mu0 + K @ (z - mu0))).max() < 2e-3
    assert np.abs(S - (np.eye(n) - K) @ cov0).max() < 5e-3


def test_P10b_partial_state_correction_direct_and_kalman():
    """f2: y = H x + v with the paper's single-state measurement (y = x3) and a 2 x 3 H.
    Direct definition of Eq. (4), Kalman posterior on the grid, and H = I reduces to correct()."""
    n, dx = 3, 0.2
    mu0, cov0 = np.array([-11.5, -10, 9.5]), np.array([[1.0, 0.3, 0.0], [0.3, 0.5, -0.1], [0.0, -0.1, 0.8]])
    for H, y, R in [(np.array([[0.0, 0.0, 1.0]]), np.array([9.1]), np.array([[1.0]])),
                    (np.array([[1.0, 0.0, 0.5], [0.0, 2.0, -1.0]]), np.array([-6.9, -29.2]), np.array([[0.9, 0.2], [0.2, 1.4]]))]:
        o = Oracle(n, [dx] * n, 1e-9, 0, [10, 8 / 3, 28])
        o.init_gaussian(mu0, cov0)
        keys, p0 = o.export()
        o.correct_linear(H, y, R)
        k1, p1 = o.export()
        assert np.array_equal(keys, k1)
        x = mu0 + keys * dx
        d = y - x @ H.T
        L = np.exp(-0.5 * np.einsum("ij,jk,ik->i", d, np.linalg.inv(R), d))
        want = p0 * L / (p0 * L).sum()
        assert np.max(np.abs(p1 - want)) <= 1e-13 * want.max()
        K = cov0 @ H.T @ np.linalg.inv(H @ cov0 @ H.T + R)
        m, S = _moments(keys, p1, mu0, np.array([dx] * n))
        assert np.abs(m - (mu0 + K @ (y - H @ mu0))).max() < 3e-3
        assert np.abs(S - (np.eye(n) - K @ H) @ cov0).max() < 6e-3
    # H = I: identical to the full-state correction
    z, R = np.array([-11.0, -10.4, 9.9]), np.array([[1.0, 0.2, 0], [0.2, 0.7, 0.1], [0, 0.1, 1.2]])
    a = Oracle(n, [dx] * n, 1e-9, 0, [10, 8 / 3, 28]); a.init_gaussian(mu0, cov0); a.correct(z, R)
    b = Oracle(n, [dx] * n, 1e-9, 0, [10, 8 / 3, 28]); b.init_gaussian(mu0, cov0); b.correct_linear(np.eye(3), z, R)
    assert np.array_equal(a.export()[1], b.export()[1])


def test_P10c_range_measurement_direct_and_1d_reduction():
    """f2, non-linear h(x) = ||x - s||: direct definition of Eq. (4); in 1-D with s far to the left the range
    is x - s, so the update equals the linear one with H = (1), y' = y + s; the posterior concentrates on
    the sphere of radius y (mean range -> y as sigma -> 0)."""
    n, dx = 3, 0.25
    mu0, cov0 = np.array([1.0, -2.0, 0.5]), np.diag([1.0, 0.6, 0.8])
    s0, y, sig = np.array([-1.0, 0.5, 0.0]), 3.2, 0.4
    o = Oracle(n, [dx] * n, 1e-9, 4, [0.0] * n)
    o.init_gaussian(mu0, cov0)
    keys, p0 = o.export()
    o.correct_range(s0, y, sig)
    k1, p1 = o.export()
    r = np.linalg.norm(mu0 + keys * dx - s0, axis=1)
    L = np.exp(-0.5 * ((y - r) / sig) ** 2)
    want = p0 * L / (p0 * L).sum()
    assert np.array_equal(keys, k1) and np.max(np.abs(p1 - want)) <= 1e-13 * want.max()
    o2 = Oracle(n, [dx] * n, 1e-9, 4, [0.0] * n); o2.init_gaussian(mu0, cov0); o2.correct_range(s0, y, 0.05)
    k2, p2 = o2.export()
    assert abs((p2 * np.linalg.norm(mu0 + k2 * dx - s0, axis=1)).sum() - y) < 0.02
    a = Oracle(1, [0.1], 1e-9, 4, [0.0]); a.init_gaussian([0.3], [[0.5]]); a.correct_range([-50.0], 50.9, 0.3)
    b = Oracle(1, [0.1], 1e-9, 4, [0.0]); b.init_gaussian([0.3], [[0.5]]); b.correct_linear([[1.0]], [0.9], [[0.09]])
    assert np.max(np.abs(a.export()[1] - b.export()[1])) <= 1e-12


def test_A8_init_gaussian_set_and_values():
    n, dx, thr = 3, 0.5, 2e-5
    cov = np.array([[1.0, 0.3, 0.0], [0.3, 0.8, -0.2], [0.0, -0.2, 1.1]])
    o = Oracle(n, [dx] * n, thr, 0, [10, 8 / 3, 28])
    o.init_gaussian([-11.5, -10, 9.5], cov)
    keys, p = o.export()
    cand = box([-14] * 3, [15] * 3)
    d = cand * dx
    g = np.exp(-0.5 * np.einsum("ij,jk,ik->i", d, np.linalg.inv(cov), d)) * dx ** 3 / np.sqrt(
        (2 * np.pi) ** 3 * np.linalg.det(cov))
    sel = g >= thr
    assert np.array_equal(keys, cand[sel])
    assert np.max(np.abs(p - g[sel] / g[sel].sum())) < 1e-15
    # BASELINE config 0 / config 2 initial sets (sizes quoted in SURVEY.md 8(a))
    o.init_gaussian([-11.5, -10, 9.5], np.eye(3))
    assert o.count() == 1357


# ---- P12 grow / prune duality (independent python statement of Targets, D1.1 / D3) ------------------------
def py_targets(c, dyn, params, origin, h):
    n = len(c)

    def u(cell, j):
        x = [np.float64(origin[m] + (cell[m] - (0.5 if m == j else 0.0)) * h[m]) for m in range(n)]
        return float(dense_ctu.dynamics(dyn, params, x, j))

    out = {}
    for j in range(n):
        up = list(c)
        up[j] += 1
        if u(up, j) > 0:
            out[j] = out.get(j, []) + [+1]
        if u(c, j) < 0:
            out[j] = out.get(j, []) + [-1]
    tg = set()
    for j, ss in out.items():
        for s in ss:
            t = list(c); t[j] += s; tg.add(tuple(t))
            for l, sl in out.items():
                if l > j:
                    for s2 in sl:
                        t2 = list(t); t2[l] += s2; tg.add(tuple(t2))
    return tg


@pytest.mark.parametrize("n,dyn,params,mean,cov,dx,thr", [
    (3, 0, [10, 8 / 3, 28], [-11.5, -10, 9.5], 1.0, 0.5, 2e-5),
    (4, 2, [4.0], [4.01, 4, 4, 4], 0.25, 0.5, 1e-5),
])
def test_P12_grow_prune_duality(n, dyn, params, mean, cov, dx, thr):
    h = [dx] * n
    o = Oracle(n, h, thr, dyn, params)
    o.init_gaussian(mean, cov * np.eye(n))
    for it in range(3):
        k0, p0 = o.export()
        o.step()
        k1, p1 = o.export()
        set1 = set(map(tuple, k1.tolist()))
        assert len(set1) == len(k1)                      # no key twice
        want = set(map(tuple, k0.tolist()))
        for c in k0[p0 >= thr].tolist():
            tg = py_targets(c, dyn, params, mean, h)
            assert tg == set(map(tuple, o.targets(c).tolist()))
            want |= tg
        assert set1 == want                              # grow = exactly I u Targets(S)
        o.prune()
        k2, p2 = o.export()
        keep = set()
        for c in k1[p1 >= thr].tolist():
            keep.add(tuple(c))
            keep |= py_targets(c, dyn, params, mean, h) & set1
        assert set(map(tuple, k2.tolist())) == keep      # D3
        assert p2.sum() == pytest.approx(1.0, abs=1e-13)
        o.prune()
        k3, _ = o.export()
        assert np.array_equal(k2, k3)                    # prune is idempotent


# ---- P13 reflection symmetry -------------------------------------------------------------------------------
@pytest.mark.parametrize("axis", [0, 1, 2])
def test_P13_reflection(axis):
    rng = np.random.default_rng(S0 + 113)
    n, A = 3, rng.normal(0, 0.5, (3, 3))
    h, origin = np.array([0.5, 0.4, 0.3]), np.array([0.2, -0.1, 0.3])
    keys = box([-3] * 3, [4] * 3)
    keys = keys[rng.random(len(keys)) < 0.7]
    p = rng.random(len(keys))
    M = np.eye(3); M[axis, axis] = -1
    o1 = raw(n, h, 3, A.ravel(), keys, p, origin=origin)
    o2 = raw(n, h, 3, (M @ A @ M).ravel(), keys * M.diagonal().astype(np.int32), p, origin=M @ origin)
    # Eq. (8) as printed uses the LOWER faces only (reading A4), which a reflection maps to upper
    # faces: dt itself is not mirror-symmetric, so both runs take the same capped step.
    for _ in range(2):
        assert o1.step(0.05) == 0.05 and o2.step(0.05) == 0.05
    k1, p1 = o1.export(); k2, p2 = o2.export()
    d1 = as_dict(k1, p1)
    d2 = as_dict(k2 * M.diagonal().astype(np.int32), p2)
    assert d1.keys() == d2.keys()
    assert max(abs(d1[k] - d2[k]) for k in d1) <= 1e-14 * p1.max()


def test_F1_metrics_oracle_pins():
    """BC (Eq. 9) and the 1-norm E: identical -> (1, 0), disjoint -> (0, 2), and two
    discretised 1-D Gaussians N(0, s^2), N(d, s^2): BC -> exp(-d^2 / (8 s^2)), E -> 2 (2 Phi(d / 2s) - 1)."""
    from math import erf, exp, sqrt
    from oracle import metrics_oracle as M
    h, s, d = 0.01, 1.0, 0.7
    k = np.arange(-900, 1000)[:, None]
    x = k[:, 0] * h
    pa = np.exp(-0.5 * (x / s) ** 2); pa /= pa.sum()
    pb = np.exp(-0.5 * ((x - d) / s) ** 2); pb /= pb.sum()
    assert M.bc_and_l1(k, pa, k, pa) == (pytest.approx(1.0, abs=1e-12), 0.0)
    assert M.bc_and_l1(k, pa, k + 5000, pa) == (0.0, pytest.approx(2.0, abs=1e-12))
    bc, l1 = M.bc_and_l1(k, pa, k, pb)
    assert bc == pytest.approx(exp(-d * d / (8 * s * s)), abs=1e-6)
    assert l1 == pytest.approx(2 * (2 * 0.5 * (1 + erf(d / (2 * s) / sqrt(2))) - 1), abs=1e-4)
    # partially overlapping key sets: cells present on one side only count with probability 0 on the other
    ka, kb = np.array([[0], [1], [2]]), np.array([[1], [2], [3]])
    bc, l1 = M.bc_and_l1(ka, np.array([0.5, 0.25, 0.25]), kb, np.array([0.25, 0.25, 0.5]))
    assert bc == pytest.approx(sqrt(0.25 * 0.25) + 0.25) and l1 == pytest.approx(0.5 + 0.0 + 0.0 + 0.5)


def test_F3_marginal_oracle_pins():
    """Marginals: mass is preserved, the marginal of a product measure is its factor,
    and integrating out nothing / everything gives the PDF itself / the total mass."""
    from oracle import marginal_oracle as MO
    rng = np.random.default_rng(5)
    a, b, c = rng.random(5), rng.random(4), rng.random(3)
    keys = np.array([[i, j, k] for i in range(5) for j in range(4) for k in range(3)], dtype=np.int32) - 2
    p = np.array([a[i] * b[j] * c[k] for i in range(5) for j in range(4) for k in range(3)])
    k1, m1 = MO.marginal(keys, p, [1])
    assert np.array_equal(k1[:, 0], np.arange(4) - 2) and np.allclose(m1, b * a.sum() * c.sum(), rtol=1e-14)
    k02, m02 = MO.marginal(keys, p, [2, 0])                 # kept dims in the order asked for
    want = {(k - 2, i - 2): c[k] * a[i] * b.sum() for i in range(5) for k in range(3)}
    assert all(abs(want[tuple(kk)] - v) < 1e-14 for kk, v in zip(k02.tolist(), m02.tolist())) and len(k02) == 15
    assert m02.sum() == pytest.approx(p.sum(), rel=1e-14)
    kall, mall = MO.marginal(keys, p, [0, 1, 2])
    assert np.array_equal(kall, keys) and np.array_equal(mall, p)


def test_F1b_resample_oracle_pins():
    """Conservative remap between grids of different spacing (reading A19; spatial convergence):
    mass is preserved, the same grid gives the same PDF, a product measure remaps factor by factor, a 3:1
    nested grid is the plain sum over the 3^n children, and a uniform density stays uniform."""
    from oracle import resample_oracle as RO
    rng = np.random.default_rng(S0 + 401)
    # (1) mass, (2) identity
    keys = box([-3, -2, -4], [4, 3, 2])
    keys = keys[rng.random(len(keys)) < 0.7]
    p = rng.random(len(keys)) - 0.1                                    # negatives are kept (A5)
    o, h = np.array([0.3, -1.0, 2.0]), np.array([0.5, 0.25, 0.4])
    o2, h2 = np.array([0.1, -0.9, 2.3]), np.array([0.8, 0.3, 0.4])
    k2, p2 = RO.resample(keys, p, o, h, o2, h2)
    assert p2.sum() == pytest.approx(p.sum(), rel=1e-13)
    ks, ps = RO.resample(keys, p, o, h, o, h)
    order = np.lexsort(keys.T[::-1])
    assert np.array_equal(ks, keys[order]) and np.allclose(ps, p[order], rtol=1e-15, atol=0)
    # (3) product measure: remap of a product = product of the 1-D remaps
    a, b = rng.random(7), rng.random(5)
    kk = np.array([[i, j] for i in range(7) for j in range(5)], dtype=np.int32) - 2
    pp = np.array([a[i] * b[j] for i in range(7) for j in range(5)])
    oo, hh, oo2, hh2 = np.array([0.0, 1.0]), np.array([0.5, 0.5]), np.array([0.2, 1.0]), np.array([0.8, 1.25])
    k2d, p2d = RO.resample(kk, pp, oo, hh, oo2, hh2)
    ka, pa = RO.resample(np.arange(7).reshape(-1, 1) - 2, a, oo[:1], hh[:1], oo2[:1], hh2[:1])
    kb, pb = RO.resample(np.arange(5).reshape(-1, 1) - 2, b, oo[1:], hh[1:], oo2[1:], hh2[1:])
    want = {(int(x), int(y)): u * v for x, u in zip(ka[:, 0], pa) for y, v in zip(kb[:, 0], pb)}
    assert len(k2d) == len(want)
    assert all(abs(want[tuple(k)] - v) <= 1e-14 for k, v in zip(k2d.tolist(), p2d.tolist()))
    # (4) nested 3:1 grid with a common origin: coarse cell d = sum of the fine cells 3d-1, 3d, 3d+1 per dimension
    kf = box([-4, -4], [5, 5])
    pf = rng.random(len(kf))
    kc, pc = RO.resample(kf, pf, np.zeros(2), np.array([0.2, 0.2]), np.zeros(2), np.array([0.6, 0.6]))
    lut = {tuple(k): v for k, v in zip(kf.tolist(), pf.tolist())}
    for d, v in zip(kc.tolist(), pc.tolist()):
        s = sum(lut.get((3 * d[0] + i, 3 * d[1] + j), 0.0) for i in (-1, 0, 1) for j in (-1, 0, 1))
        assert v == pytest.approx(s, rel=1e-13)
    assert len(kc) == 9
    # (5) 1-D uniform density rho on cells -10..10 (h = 0.3): interior cells of the h2 = 0.7 grid get rho * h2
    k1 = np.arange(-10, 11).reshape(-1, 1).astype(np.int32)
    kq, pq = RO.resample(k1, np.full(21, 2.0 * 0.3), np.array([0.05]), np.array([0.3]), np.array([0.0]), np.array([0.7]))
    inner = np.abs(kq[:, 0]) <= 3
    assert np.allclose(pq[inner], 2.0 * 0.7, rtol=1e-13)
