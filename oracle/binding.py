"""ctypes binding to the serial C++ oracle (gbeeso_* C ABI). Test infrastructure only."""
import ctypes as C

import numpy as np

from . import build as _build

_lib = None


def lib():
    global _lib
    if _lib is None:
        L = C.CDLL(_build.build())
        dp, ip, vp = C.POINTER(C.c_double), C.POINTER(C.c_int32), C.c_void_p
        L.gbeeso_create.argtypes = [C.POINTER(vp), C.c_int, dp, C.c_double, C.c_int, dp, C.c_int,
                                    C.c_double, C.c_int, C.c_int]
        L.gbeeso_destroy.argtypes = [vp]
        L.gbeeso_set_flags.argtypes = [vp, C.c_int, C.c_int]
        L.gbeeso_init_gaussian.argtypes = [vp, dp, dp]
        L.gbeeso_import.argtypes = [vp, dp, ip, dp, C.c_int64]
        L.gbeeso_step.argtypes = [vp, dp]
        L.gbeeso_prune.argtypes = [vp]
        L.gbeeso_correct.argtypes = [vp, dp, dp]
        L.gbeeso_correct_linear.argtypes = [vp, dp, C.c_int, dp, dp]
        L.gbeeso_correct_range.argtypes = [vp, dp, C.c_double, C.c_double]
        L.gbeeso_export.argtypes = [vp, ip, dp, C.c_int64, C.POINTER(C.c_int64)]
        L.gbeeso_count.argtypes = [vp]
        L.gbeeso_count.restype = C.c_int64
        for f in (L.gbeeso_time, L.gbeeso_last_mass, L.gbeeso_last_dt):
            f.argtypes = [vp]
            f.restype = C.c_double
        L.gbeeso_face_velocity.argtypes = [vp, ip, C.c_int]
        L.gbeeso_face_velocity.restype = C.c_double
        L.gbeeso_targets.argtypes = [vp, ip, ip]
        L.gbeeso_dynamics.argtypes = [vp, dp, dp]
        L.gbeeso_ht_lookup.argtypes = [C.POINTER(C.c_uint64), C.c_int64, C.POINTER(C.c_uint64),
                                       C.c_int64, C.POINTER(C.c_uint8)]
        _lib = L
    return _lib


def _d(a):
    a = np.ascontiguousarray(a, dtype=np.float64)
    return a, a.ctypes.data_as(C.POINTER(C.c_double))


def _i(a):
    a = np.ascontiguousarray(a, dtype=np.int32)
    return a, a.ctypes.data_as(C.POINTER(C.c_int32))


class OracleError(RuntimeError):
    pass


def _chk(rc, what):
    if rc != 0:
        raise OracleError(f"oracle {what} failed rc={rc}")


class Oracle:
    """Serial CPU GBEES (same call sequence as the product's Gbees class)."""

    def __init__(self, n, dx, threshold, dynamics_id, params, cfl=0.9, hi_res=1, limiter=0):
        self.n = int(n)
        self._h = C.c_void_p()
        _, dxp = _d(dx)
        par, pp = _d(params)
        _chk(lib().gbeeso_create(C.byref(self._h), self.n, dxp, float(threshold), int(dynamics_id),
                                 pp, int(par.size), float(cfl), int(hi_res), int(limiter)), "create")

    def __del__(self):
        if getattr(self, "_h", None):
            lib().gbeeso_destroy(self._h)
            self._h = None

    def set_flags(self, grow=True, normalise=True):
        lib().gbeeso_set_flags(self._h, int(grow), int(normalise))

    def init_gaussian(self, mean, cov):
        _, m = _d(mean)
        _, c = _d(cov)
        _chk(lib().gbeeso_init_gaussian(self._h, m, c), "init_gaussian")

    def import_state(self, origin, keys, p):
        keys = np.ascontiguousarray(keys, dtype=np.int32).reshape(-1, self.n)
        _, o = _d(origin)
        _, k = _i(keys)
        pa, pp = _d(p)
        _chk(lib().gbeeso_import(self._h, o, k, pp, int(pa.size)), "import")

    def step(self, dt_cap=0.0):
        dt = C.c_double(float(dt_cap))
        _chk(lib().gbeeso_step(self._h, C.byref(dt)), "step")
        return dt.value

    def prune(self):
        _chk(lib().gbeeso_prune(self._h), "prune")

    def correct(self, z, R):
        _, zp = _d(z)
        _, rp = _d(R)
        _chk(lib().gbeeso_correct(self._h, zp, rp), "correct")

    def correct_linear(self, H, y, R):
        """Eq. (4) with y = H x + v (H m x n row-major, R m x m)."""
        Ha, hp = _d(H)
        ya, yp = _d(y)
        _, rp = _d(R)
        _chk(lib().gbeeso_correct_linear(self._h, hp, int(ya.size), yp, rp), "correct_linear")

    def correct_range(self, s, y, sigma):
        """Eq. (4) with the non-linear range measurement y = ||x - s|| + v, v ~ N(0, sigma^2)."""
        _, sp = _d(s)
        _chk(lib().gbeeso_correct_range(self._h, sp, float(y), float(sigma)), "correct_range")

    def count(self):
        return int(lib().gbeeso_count(self._h))

    def time(self):
        return float(lib().gbeeso_time(self._h))

    def last_mass(self):
        return float(lib().gbeeso_last_mass(self._h))

    def export(self, sort=True):
        N = self.count()
        keys = np.empty((N, self.n), dtype=np.int32)
        p = np.empty(N, dtype=np.float64)
        cnt = C.c_int64()
        _chk(lib().gbeeso_export(self._h, keys.ctypes.data_as(C.POINTER(C.c_int32)),
                                 p.ctypes.data_as(C.POINTER(C.c_double)), N, C.byref(cnt)), "export")
        if sort and N:
            order = np.lexsort(keys.T[::-1])
            keys, p = keys[order], p[order]
        return keys, p

    def face_velocity(self, coords, j):
        _, c = _i(coords)
        return float(lib().gbeeso_face_velocity(self._h, c, int(j)))

    def dynamics(self, x):
        """f(x) at an arbitrary point (test hook for the dynamics pins)."""
        xa, xp = _d(x)
        out = np.zeros(self.n)
        lib().gbeeso_dynamics(self._h, xp, out.ctypes.data_as(C.POINTER(C.c_double)))
        return out

    def targets(self, coords):
        _, c = _i(coords)
        out = np.zeros((72, self.n), dtype=np.int32)
        k = lib().gbeeso_targets(self._h, c, out.ctypes.data_as(C.POINTER(C.c_int32)))
        return out[:k].copy()


def ht_lookup(keys, query):
    keys = np.ascontiguousarray(keys, dtype=np.uint64)
    query = np.ascontiguousarray(query, dtype=np.uint64)
    found = np.zeros(query.size, dtype=np.uint8)
    u64p = C.POINTER(C.c_uint64)
    lib().gbeeso_ht_lookup(keys.ctypes.data_as(u64p), keys.size, query.ctypes.data_as(u64p),
                           query.size, found.ctypes.data_as(C.POINTER(C.c_uint8)))
    return found.astype(bool)
