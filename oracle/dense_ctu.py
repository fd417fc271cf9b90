"""Dense-array CTU checker (numpy) -- TEST INFRASTRUCTURE ONLY.

A second, independent statement of one flux+update pass, in the *gather / predictor* form D2 of
SURVEY.md section 8(c) (the C++ oracle uses the scatter form D1.3 = Eq. (7) + Algorithm 1 of
PAPER.md:79-110). Used for pin P7: brute-force agreement between the two forms on tiny boxes with
an arbitrary `active` mask, and by P3/P13. Everything lives on a dense padded box; P reads as 0
and `active` as False outside the stored cells (reading A6).

    T_{c,l}   = u+_{c,l} (P_c - P_{c-e^l}) + u-_{c+e^l,l} (P_{c+e^l} - P_c)        (c active, else 0)
    P*_{c,(j)} = P_c - sum_{l != j} 1/2 tau_l T_{c,l}                               (c active, else 0)
    F(c,j)    = u+_{c,j} P*_{c-e^j,(j)} + u-_{c,j} P*_{c,(j)} + 1/2 |u| (1 - tau_j |u|) W~
    P'_c      = P_c - sum_j tau_j (F(c+e^j,j) - F(c,j))                             (c active)
"""
import numpy as np

PAD = 3


def _at(A, j, s):
    """Array whose entry at c is A[c + s e^j] (padding keeps the wrap-around out of reach)."""
    return np.roll(A, -s, axis=j)


def dynamics(dyn, params, x, j):
    """f_j evaluated on arrays of coordinates x[0..n-1] (same formulas as PAPER.md:303/319)."""
    n = len(x)
    p = np.asarray(params, dtype=np.float64)
    if dyn == 0:
        return [p[0] * (x[1] - x[0]), x[0] * (p[2] - x[2]) - x[1], x[0] * x[1] - p[1] * x[2]][j]
    if dyn == 1:
        return [p[0] * (x[1] - x[0]), -x[1] - x[0] * x[2], x[0] * x[1] - p[1] * x[2] - p[1] * p[2]][j]
    if dyn == 2:
        return (x[(j + 1) % n] - x[(j - 2) % n]) * x[(j - 1) % n] - x[j] + p[0]
    if dyn == 3:
        A = p.reshape(n, n)
        return sum(A[j, m] * x[m] for m in range(n))
    if dyn == 4:
        return np.full_like(x[0], p[j])
    raise ValueError(dyn)


def face_velocities(dyn, params, origin, h, lo, shape):
    """U[j][c] = f_j at the lower j-face of cell c, for every c of the box [lo, lo+shape)."""
    n = len(shape)
    idx = np.meshgrid(*[np.arange(lo[m], lo[m] + shape[m], dtype=np.float64) for m in range(n)],
                      indexing="ij")
    U = []
    for j in range(n):
        x = [origin[m] + (idx[m] - (0.5 if m == j else 0.0)) * h[m] for m in range(n)]
        U.append(dynamics(dyn, params, x, j))
    return U


def mc(a, b):
    m = np.minimum(0.5 * np.abs(a + b), np.minimum(2.0 * np.abs(a), 2.0 * np.abs(b)))
    return np.where(a * b <= 0.0, 0.0, np.sign(a) * m)


def dense_step(P, active, U, dt, h, hi_res=True, limiter=0):
    """One un-normalised flux+update pass on a dense padded box. Returns P' (0 off `active`)."""
    n = P.ndim
    act = active.astype(np.float64)
    P = P * act
    tau = [dt / h[j] for j in range(n)]
    up = [np.maximum(U[j], 0.0) for j in range(n)]
    um = [np.minimum(U[j], 0.0) for j in range(n)]
    T = []
    for l in range(n):
        T.append(act * (up[l] * (P - _at(P, l, -1)) + _at(um[l], l, +1) * (_at(P, l, +1) - P)))
    Pn = P.copy()
    for j in range(n):
        Ps = P.copy()
        for l in range(n):
            if l != j:
                Ps = Ps - 0.5 * tau[l] * T[l]
        Ps = Ps * act
        F = up[j] * _at(Ps, j, -1) + um[j] * Ps
        if hi_res:
            W = P - _at(P, j, -1)
            if limiter == 1:
                Wl = W
            else:
                Wup = np.where(U[j] > 0.0, _at(P, j, -1) - _at(P, j, -2), _at(P, j, +1) - P)
                Wl = mc(W, Wup)
            au = np.abs(U[j])
            F = F + 0.5 * au * (1.0 - tau[j] * au) * Wl
        Pn = Pn - tau[j] * (_at(F, j, +1) - F)
    return Pn * act


def to_dense(keys, p, pad=PAD):
    """Scatter a sparse state (int coords [N,n], values [N]) onto a dense padded box."""
    keys = np.asarray(keys)
    lo = keys.min(axis=0) - pad
    shape = tuple((keys.max(axis=0) - keys.min(axis=0) + 1 + 2 * pad).tolist())
    P = np.zeros(shape)
    act = np.zeros(shape, dtype=bool)
    ix = tuple((keys - lo).T)
    P[ix] = p
    act[ix] = True
    return P, act, lo, shape


def dense_step_sparse(keys, p, dyn, params, origin, h, dt, hi_res=True, limiter=0):
    """Dense step of a sparse state; returns P' gathered back at `keys` (un-normalised)."""
    P, act, lo, shape = to_dense(keys, p)
    U = face_velocities(dyn, params, origin, h, lo, shape)
    Pn = dense_step(P, act, U, dt, h, hi_res, limiter)
    return Pn[tuple((np.asarray(keys) - lo).T)]
