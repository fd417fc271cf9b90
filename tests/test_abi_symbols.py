"""The C-ABI library loads on a CPU-only box and exports every symbol include/gbees.h declares."""
import ctypes
import os
import re

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def declared_symbols():
    src = open(os.path.join(ROOT, "include", "gbees.h")).read()
    src = re.sub(r"/\*.*?\*/", "", src, flags=re.S)
    return sorted(set(re.findall(r"\b(gbees_[a-z0-9_]+)\s*\(", src)))


def test_library_exports_every_declared_symbol():
    from paper_2508_13986_b200 import build, binding
    build.build()
    L = ctypes.CDLL(binding.lib_path())
    names = declared_symbols()
    assert {"gbees_create", "gbees_init_gaussian", "gbees_step", "gbees_prune", "gbees_correct",
            "gbees_export", "gbees_run"} <= set(names)
    missing = [n for n in names if not hasattr(L, n)]
    assert not missing, missing


def test_default_opts_and_argument_checks_without_gpu():
    from paper_2508_13986_b200 import binding
    L = binding.lib()
    o = binding.Opts()
    assert L.gbees_default_opts(ctypes.byref(o)) == 0
    assert (o.max_cells, o.load_factor, o.cfl, o.hi_res, o.limiter) == (1 << 20, 0.5, 0.9, 1, 0)
    h = ctypes.c_void_p()
    dx = (ctypes.c_double * 3)(0.5, 0.5, 0.5)
    par = (ctypes.c_double * 3)(10, 8 / 3, 28)
    assert L.gbees_create(ctypes.byref(h), 7, dx, 1e-5, 0, par, 3, None) == -1      # n out of range
    assert L.gbees_create(ctypes.byref(h), 3, dx, 1e-5, 2, par, 3, None) == -1      # Lorenz '96 needs n >= 4
    assert L.gbees_create(ctypes.byref(h), 3, dx, 1e-5, 0, par, 2, None) == -1      # too few params


def test_arena_bytes_without_gpu():
    """caller-provided device arena; its size is a host-side function of (n, max_cells, load_factor)."""
    from paper_2508_13986_b200 import binding
    small, big = binding.arena_bytes(6, 1 << 16), binding.arena_bytes(6, 1 << 22)
    assert 0 < small < big
    # dominated by the bricks: 2 x 512 (Q, Qn) + 2n x 256 (phi) bytes per brick, max_cells / 16 bricks
    bricks = (1 << 22) // 16
    assert big >= bricks * (1024 + 12 * 256) and big < 2 * bricks * (1024 + 12 * 256)
    assert binding.arena_bytes(3, 1 << 22) < big                       # fewer faces per brick
    b = ctypes.c_int64()
    assert binding.lib().gbees_arena_bytes(7, None, ctypes.byref(b)) == -1


def test_product_does_not_import_oracle():
    pkg = os.path.join(ROOT, "paper_2508_13986_b200")
    for dirpath, _, files in os.walk(pkg):
        for f in files:
            if f.endswith((".py", ".cu", ".cuh", ".h")):
                txt = open(os.path.join(dirpath, f)).read()
                assert not re.search(r"import\s+oracle|from\s+oracle|libgbees_oracle|gbeeso_|oracle/", txt), f
