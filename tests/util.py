"""Comparison helpers for GPU-vs-oracle parity (north_star tolerances, readings A14/A15)."""
import numpy as np


def key_set(keys):
    return set(map(tuple, keys.tolist()))


def compare_states(gk, gp, ok, op, thresh, rtol, band=1e-12, what=""):
    """Active sets identical, except (reading A14) zero-mass cells next to a cell whose mass lies within `band`
    (relative) of the threshold: such a cell may flip its source status in one of the two runs, and its targets
    -- face or pairwise-edge neighbours, i.e. cells at Chebyshev distance 1 -- then exist on one side only.
    Probabilities within rtol relative in max-norm over the common cells."""
    if gk.shape == ok.shape and np.array_equal(gk, ok):
        pass
    else:
        gs, os_ = key_set(gk), key_set(ok)
        od = {tuple(k): v for k, v in zip(ok.tolist(), op.tolist())}
        gd = {tuple(k): v for k, v in zip(gk.tolist(), gp.tolist())}
        n = gk.shape[1]
        for k in gs ^ os_:
            v = od.get(k, gd.get(k))
            assert v == 0.0, f"{what}: key {k} only on one side with P = {v}"
            # a parent in the band: some cell at Chebyshev distance 1 (in either state) with |P / p* - 1| < band
            near = False
            for d in np.ndindex(*([3] * n)):
                c = tuple(int(k[j] + d[j] - 1) for j in range(n))
                for st in (od, gd):
                    pv = st.get(c)
                    if pv is not None and thresh > 0 and abs(pv / thresh - 1.0) < band:
                        near = True
            assert near, f"{what}: key {k} only on one side (P = 0) and no neighbouring cell within {band} of the threshold"
        common = sorted(gs & os_)
        gp = np.array([gd[k] for k in common])
        op = np.array([od[k] for k in common])
    err = np.max(np.abs(gp - op)) / np.max(np.abs(op))
    assert err <= rtol, f"{what}: max-norm relative error {err:.3e} > {rtol:.1e}"
    return err


def sort_state(keys, p):
    """Lexicographic order (dimension 0 most significant) through one packed int64 key per cell
    (10 bits per coordinate for n = 6, i.e. |c| < 512: the packable range of the product itself)."""
    keys = np.ascontiguousarray(keys, dtype=np.int32)
    n = keys.shape[1]
    bits = 63 // n if 63 // n < 31 else 31
    code = np.zeros(len(keys), dtype=np.int64)
    for j in range(n):
        code = (code << bits) | (keys[:, j].astype(np.int64) + (1 << (bits - 1)))
    order = np.argsort(code, kind="stable")
    return np.ascontiguousarray(keys[order]), np.asarray(p)[order]


def key_hash(keys_sorted):
    """sha256 of the sorted int32 key array (bit-exact active-set fingerprint)."""
    import hashlib
    return hashlib.sha256(np.ascontiguousarray(keys_sorted, dtype=np.int32).tobytes()).hexdigest()
