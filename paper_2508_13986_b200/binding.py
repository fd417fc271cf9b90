"""ctypes binding with the same names as include/gbees.h (argument marshalling only)."""
import ctypes as C
import os

import numpy as np

HERE = os.path.dirname(os.path.abspath(__file__))
_LIB_PATH = os.path.join(HERE, "libgbees.so")
_lib = None

ERRORS = {-1: "ARG", -2: "CUDA", -3: "NOT_SPD", -4: "CAPACITY", -5: "BUFFER", -6: "DEGENERATE", -7: "KEY_RANGE"}


class GbeesError(RuntimeError):
    def __init__(self, code, msg):
        super().__init__(f"gbees error {code} ({ERRORS.get(code, '?')}): {msg}")
        self.code = code


class Opts(C.Structure):
    _fields_ = [("max_cells", C.c_int64), ("load_factor", C.c_double), ("cfl", C.c_double),
                ("hi_res", C.c_int), ("limiter", C.c_int), ("no_grow", C.c_int), ("no_normalise", C.c_int),
                ("run_mode", C.c_int), ("device", C.c_int), ("stream", C.c_void_p), ("arena", C.c_void_p), ("arena_bytes", C.c_int64)]


class Stats(C.Structure):
    _fields_ = [("n_cells", C.c_int64), ("n_inserted", C.c_int64), ("n_pruned", C.c_int64), ("steps", C.c_int64),
                ("t", C.c_double), ("dt", C.c_double), ("mass", C.c_double), ("cell_updates", C.c_int64),
                ("table_slots", C.c_int64), ("launches", C.c_int64),
                ("cells_inserted", C.c_int64), ("cells_prune_scanned", C.c_int64), ("prunes", C.c_int64)]

PHASES = ["grow", "link", "passA", "passB", "mark", "compact", "rebuild", "relink", "sum", "correct", "run"]


def arena_bytes(n, max_cells=1 << 20, load_factor=0.5):
    """Device bytes a context of this capacity carves from a caller-provided arena (gbees_arena_bytes)."""
    o = Opts()
    lib().gbees_default_opts(C.byref(o))
    o.max_cells, o.load_factor = int(max_cells), float(load_factor)
    b = C.c_int64()
    rc = lib().gbees_arena_bytes(int(n), C.byref(o), C.byref(b))
    if rc:
        raise GbeesError(rc, "gbees_arena_bytes failed")
    return b.value


NOALLOC_MAX_CELLS = 131072   # GBEES_NOALLOC_MAX_CELLS in include/gbees.h


def marginal_noalloc(keys_t, p_t, dims, out_keys_t, out_p_t, device=0, stream=None):
    """gbees_marginal_noalloc: marginal of an exported state held in torch CUDA tensors (keys int32 [N, n],
    p float64 [N]) into caller-owned CUDA tensors (int32 [cap, m], float64 [cap]); nothing is allocated.
    Returns the number of marginal cells written."""
    d = (C.c_int * len(dims))(*[int(x) for x in dims])
    cnt = C.c_int64()
    rc = lib().gbees_marginal_noalloc(int(device), C.c_void_p(stream) if stream else None, int(keys_t.shape[1]),
                                      keys_t.data_ptr(), p_t.data_ptr(), int(p_t.numel()), d, len(dims),
                                      out_keys_t.data_ptr(), out_p_t.data_ptr(), int(out_p_t.numel()), C.byref(cnt))
    if rc:
        raise GbeesError(rc, lib().gbees_marginal_noalloc_error().decode())
    return cnt.value


def lib_path():
    return _LIB_PATH


def lib():
    """Load libgbees.so. Fails loudly when the CUDA extension has not been built."""
    global _lib
    if _lib is None:
        if not os.path.exists(_LIB_PATH):
            raise ImportError(f"{_LIB_PATH} is missing: run `python -c 'import __graft_entry__ as g; g.build()'` "
                              "(there is no CPU fallback)")
        L = C.CDLL(_LIB_PATH)
        vp, dp, ip = C.c_void_p, C.POINTER(C.c_double), C.c_void_p
        L.gbees_default_opts.argtypes = [C.POINTER(Opts)]
        L.gbees_arena_bytes.argtypes = [C.c_int, C.POINTER(Opts), C.POINTER(C.c_int64)]
        L.gbees_create.argtypes = [C.POINTER(vp), C.c_int, dp, C.c_double, C.c_int, dp, C.c_int, C.POINTER(Opts)]
        L.gbees_destroy.argtypes = [vp]
        L.gbees_init_gaussian.argtypes = [vp, dp, dp]
        L.gbees_import.argtypes = [vp, dp, ip, C.c_void_p, C.c_int64]
        L.gbees_step.argtypes = [vp, dp]
        L.gbees_prune.argtypes = [vp]
        L.gbees_correct.argtypes = [vp, dp, dp]
        L.gbees_export.argtypes = [vp, C.c_void_p, C.c_void_p, C.c_int64, C.POINTER(C.c_int64)]
        L.gbees_run.argtypes = [vp, C.c_double, C.c_int64, C.c_int, C.POINTER(C.c_int64)]
        L.gbees_count.argtypes = [vp, C.POINTER(C.c_int64)]
        L.gbees_time.argtypes = [vp, dp]
        L.gbees_correct_linear.argtypes = [vp, dp, C.c_int, dp, dp]
        L.gbees_compare.argtypes = [vp, vp, dp, dp]
        L.gbees_correct_range.argtypes = [vp, dp, C.c_double, C.c_double]
        L.gbees_marginal.argtypes = [vp, C.POINTER(C.c_int), C.c_int, vp, vp, C.c_int64, C.POINTER(C.c_int64)]
        L.gbees_resample.argtypes = [vp, dp, dp, vp, vp, C.c_int64, C.POINTER(C.c_int64)]
        L.gbees_stats.argtypes = [vp, C.POINTER(Stats)]
        L.gbees_profile.argtypes = [vp, C.c_int, dp, C.POINTER(C.c_int64)]
        L.gbees_marginal_noalloc.argtypes = [C.c_int, vp, C.c_int, vp, vp, C.c_int64, C.POINTER(C.c_int), C.c_int, vp, vp,
                                             C.c_int64, C.POINTER(C.c_int64)]
        L.gbees_marginal_noalloc_error.restype = C.c_char_p
        L.gbees_last_error.argtypes = [vp]
        L.gbees_last_error.restype = C.c_char_p
        L.gbees_clear_error.argtypes = [vp]
        _lib = L
    return _lib


def _d(a):
    a = np.ascontiguousarray(a, dtype=np.float64)
    return a, a.ctypes.data_as(C.POINTER(C.c_double))


class Gbees:
    """One GBEES context on one GPU. Methods mirror the C ABI one to one."""

    def __init__(self, n, dx, threshold, dynamics_id, params, max_cells=1 << 20, load_factor=0.5, cfl=0.9,
                 hi_res=1, limiter=0, no_grow=False, no_normalise=False, run_mode=0, device=0, stream=None, arena=None):
        L = lib()
        self.n = int(n)
        o = Opts()
        L.gbees_default_opts(C.byref(o))
        o.max_cells, o.load_factor, o.cfl = int(max_cells), float(load_factor), float(cfl)
        o.hi_res, o.limiter, o.no_grow, o.no_normalise = int(hi_res), int(limiter), int(no_grow), int(no_normalise)
        o.device = int(device)
        o.run_mode = int(run_mode)
        o.stream = C.c_void_p(stream) if stream else None
        if arena is not None:                       # a torch CUDA uint8 tensor owned by the caller: all device structures live in it
            o.arena, o.arena_bytes = C.c_void_p(arena.data_ptr()), int(arena.numel() * arena.element_size())
            self._arena = arena
        self._h = C.c_void_p()
        _, dxp = _d(dx)
        par, pp = _d(params)
        rc = L.gbees_create(C.byref(self._h), self.n, dxp, float(threshold), int(dynamics_id), pp, int(par.size),
                            C.byref(o))
        if rc:
            self._h = None
            raise GbeesError(rc, "gbees_create failed")

    def close(self):
        if getattr(self, "_h", None):
            lib().gbees_destroy(self._h)
            self._h = None

    __del__ = close

    def _chk(self, rc):
        if rc:
            raise GbeesError(rc, lib().gbees_last_error(self._h).decode())

    def init_gaussian(self, mean, cov):
        _, m = _d(mean)
        _, c = _d(cov)
        self._chk(lib().gbees_init_gaussian(self._h, m, c))

    def import_state(self, origin, keys, p):
        """keys/p: numpy arrays (host) or torch CUDA tensors (device pointers are passed through)."""
        _, o = _d(origin)
        if hasattr(keys, "data_ptr"):
            kp, pp, cnt = keys.data_ptr(), p.data_ptr(), int(p.numel())
            hold = (keys, p)
        else:
            ka = np.ascontiguousarray(keys, dtype=np.int32).reshape(-1, self.n)
            pa = np.ascontiguousarray(p, dtype=np.float64)
            kp, pp, cnt, hold = ka.ctypes.data, pa.ctypes.data, int(pa.size), (ka, pa)
        self._chk(lib().gbees_import(self._h, o, kp, pp, cnt))
        del hold

    def step(self, dt_cap=0.0):
        dt = C.c_double(float(dt_cap))
        self._chk(lib().gbees_step(self._h, C.byref(dt)))
        return dt.value

    def prune(self):
        self._chk(lib().gbees_prune(self._h))

    def correct(self, z, R):
        _, zp = _d(z)
        _, rp = _d(R)
        self._chk(lib().gbees_correct(self._h, zp, rp))

    def correct_linear(self, H, y, R):
        Ha, hp = _d(H)
        ya, yp = _d(y)
        _, rp = _d(R)
        self._chk(lib().gbees_correct_linear(self._h, hp, int(ya.size), yp, rp))

    def correct_range(self, s, y, sigma):
        _, sp = _d(s)
        self._chk(lib().gbees_correct_range(self._h, sp, float(y), float(sigma)))

    def compare(self, other):
        """(BC, E) between this context and another one on the same grid (Eq. 9 and the 1-norm of PAPER.md:362-366)."""
        bc, l1 = C.c_double(), C.c_double()
        self._chk(lib().gbees_compare(self._h, other._h, C.byref(bc), C.byref(l1)))
        return bc.value, l1.value

    def marginal(self, dims, sort=True):
        """Host marginal over the kept dimensions `dims`: (keys int32 [M, m], p float64 [M])."""
        d = (C.c_int * len(dims))(*[int(x) for x in dims])
        cnt = C.c_int64()
        self._chk(lib().gbees_marginal(self._h, d, len(dims), None, None, 0, C.byref(cnt)))
        M = cnt.value
        keys = np.empty((M, len(dims)), dtype=np.int32)
        p = np.empty(M, dtype=np.float64)
        self._chk(lib().gbees_marginal(self._h, d, len(dims), keys.ctypes.data, p.ctypes.data, M, C.byref(cnt)))
        if sort and M:
            order = np.lexsort(keys.T[::-1])
            keys, p = keys[order], p[order]
        return keys, p

    def resample(self, origin2, dx2, sort=True):
        """Host conservative remap onto the grid (origin2, dx2): (keys int32 [M, n], p float64 [M])."""
        _, op = _d(origin2)
        _, hp = _d(dx2)
        cnt = C.c_int64()
        self._chk(lib().gbees_resample(self._h, op, hp, None, None, 0, C.byref(cnt)))
        M = cnt.value
        keys = np.empty((M, self.n), dtype=np.int32)
        p = np.empty(M, dtype=np.float64)
        self._chk(lib().gbees_resample(self._h, op, hp, keys.ctypes.data, p.ctypes.data, M, C.byref(cnt)))
        if sort and M:
            order = np.lexsort(keys.T[::-1])
            keys, p = keys[order], p[order]
        return keys, p

    def run(self, t_target, max_steps=1 << 62, prune_every=0):
        done = C.c_int64()
        self._chk(lib().gbees_run(self._h, float(t_target), int(max_steps), int(prune_every), C.byref(done)))
        return done.value

    def count(self):
        n = C.c_int64()
        self._chk(lib().gbees_count(self._h, C.byref(n)))
        return n.value

    def time(self):
        t = C.c_double()
        self._chk(lib().gbees_time(self._h, C.byref(t)))
        return t.value

    def stats(self):
        s = Stats()
        self._chk(lib().gbees_stats(self._h, C.byref(s)))
        return {k: getattr(s, k) for k, _ in Stats._fields_}

    def profile(self, enable):
        """Read-and-reset per-phase {name: (ms, launches)}, then switch event timing on/off."""
        ms = (C.c_double * len(PHASES))()
        ln = (C.c_int64 * len(PHASES))()
        self._chk(lib().gbees_profile(self._h, int(bool(enable)), ms, ln))
        return {k: (ms[i], ln[i]) for i, k in enumerate(PHASES)}

    def last_mass(self):
        return self.stats()["mass"]

    def export(self, sort=True):
        """Host export: (keys int32 [N,n], p float64 [N]); sorted lexicographically if sort."""
        N = self.count()
        keys = np.empty((N, self.n), dtype=np.int32)
        p = np.empty(N, dtype=np.float64)
        cnt = C.c_int64()
        self._chk(lib().gbees_export(self._h, keys.ctypes.data, p.ctypes.data, N, C.byref(cnt)))
        if sort and N:
            order = np.lexsort(keys.T[::-1])
            keys, p = keys[order], p[order]
        return keys, p

    def export_device(self, keys_t, p_t):
        """Device export into caller-owned torch CUDA tensors (int32 [cap,n], float64 [cap])."""
        cnt = C.c_int64()
        self._chk(lib().gbees_export(self._h, keys_t.data_ptr(), p_t.data_ptr(), int(p_t.numel()), C.byref(cnt)))
        return cnt.value


class HashTable:
    """BASELINE config 4: the library's open-addressing table on its own (gbees_ht_* in include/gbees.h).
    Keys / flags are torch CUDA tensors (int64 holding the packed 64-bit keys, uint8 delete flags)."""

    def __init__(self, slots, device=0):
        L = lib()
        vp = C.c_void_p
        L.gbees_ht_create.argtypes = [C.POINTER(vp), C.c_int64, C.c_int]
        L.gbees_ht_destroy.argtypes = [vp]
        L.gbees_ht_insert.argtypes = [vp, vp, C.c_int64, vp, C.POINTER(C.c_uint64)]
        L.gbees_ht_lookup.argtypes = [vp, vp, C.c_int64, vp, C.POINTER(C.c_uint64)]
        L.gbees_ht_compact.argtypes = [vp, vp, vp, C.c_int64, C.POINTER(C.c_int64)]
        L.gbees_ht_lookup_coop.argtypes = [vp, vp, C.c_int64, vp, C.POINTER(C.c_uint64), C.c_int]
        self._h = vp()
        rc = L.gbees_ht_create(C.byref(self._h), int(slots), int(device))
        if rc:
            self._h = None
            raise GbeesError(rc, "gbees_ht_create failed")

    def close(self):
        if getattr(self, "_h", None):
            lib().gbees_ht_destroy(self._h)
            self._h = None

    __del__ = close

    def insert(self, keys_t, idx_out_t=None):
        pr = C.c_uint64()
        rc = lib().gbees_ht_insert(self._h, keys_t.data_ptr(), int(keys_t.numel()),
                                   idx_out_t.data_ptr() if idx_out_t is not None else None, C.byref(pr))
        if rc:
            raise GbeesError(rc, "gbees_ht_insert failed")
        return pr.value

    def lookup(self, query_t, out_t=None):
        pr = C.c_uint64()
        rc = lib().gbees_ht_lookup(self._h, query_t.data_ptr(), int(query_t.numel()),
                                   out_t.data_ptr() if out_t is not None else None, C.byref(pr))
        if rc:
            raise GbeesError(rc, "gbees_ht_lookup failed")
        return pr.value

    def lookup_coop(self, query_t, out_t=None, width=4):
        pr = C.c_uint64()
        rc = lib().gbees_ht_lookup_coop(self._h, query_t.data_ptr(), int(query_t.numel()),
                                        out_t.data_ptr() if out_t is not None else None, C.byref(pr), int(width))
        if rc:
            raise GbeesError(rc, "gbees_ht_lookup_coop failed")
        return pr.value

    def compact(self, keys_t, del_t):
        k = C.c_int64()
        rc = lib().gbees_ht_compact(self._h, keys_t.data_ptr(), del_t.data_ptr(), int(keys_t.numel()), C.byref(k))
        if rc:
            raise GbeesError(rc, "gbees_ht_compact failed")
        return k.value
