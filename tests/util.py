"""Comparison helpers for GPU-vs-oracle parity (north_star tolerances, readings A14/A15)."""
import numpy as np


def key_set(keys):
    return set(map(tuple, keys.tolist()))


def compare_states(gk, gp, ok, op, thresh, rtol, band=1e-12, what=""):
    """Active sets identical except cells within `band` (relative) of the threshold and zero-mass
    cells (children of band cells); probabilities within rtol relative in max-norm."""
    if gk.shape == ok.shape and np.array_equal(gk, ok):
        common_g = common_o = slice(None)
    else:
        gs, os_ = key_set(gk), key_set(ok)
        od = {tuple(k): v for k, v in zip(ok.tolist(), op.tolist())}
        gd = {tuple(k): v for k, v in zip(gk.tolist(), gp.tolist())}
        near = any(abs(v / thresh - 1.0) < band for v in op) if thresh > 0 else False
        for k in gs ^ os_:
            v = od.get(k, gd.get(k))
            assert near and v == 0.0, f"{what}: key {k} only on one side (P={v}), no cell within the band"
        common = sorted(gs & os_)
        gp = np.array([gd[k] for k in common])
        op = np.array([od[k] for k in common])
        common_g = common_o = slice(None)
    err = np.max(np.abs(gp[common_g] - op[common_o])) / np.max(np.abs(op))
    assert err <= rtol, f"{what}: max-norm relative error {err:.3e} > {rtol:.1e}"
    return err
