"""Marginal of a grid PDF (TEST INFRASTRUCTURE ONLY): sum the cell probabilities over the dimensions
that are integrated out (the 6-D Lorenz '96 PDF is shown as two 3-D marginals).
Plain definition with numpy: group by the kept coordinates, add."""
import numpy as np


def marginal(keys, p, dims):
    sub = np.ascontiguousarray(keys[:, list(dims)])
    uniq, inv = np.unique(sub, axis=0, return_inverse=True)     # uniq is sorted lexicographically
    return uniq.astype(np.int32), np.bincount(inv.ravel(), weights=p, minlength=len(uniq))
