"""The comparison helper of the parity tests (tests/util.py, reading A14) does what it says."""
import numpy as np
import pytest

from util import compare_states


def test_compare_states_band_rule():
    thr = 1e-5
    k = np.array([[0, 0], [0, 1], [1, 0]], dtype=np.int32)
    p = np.array([0.5, 0.3, 0.2])
    assert compare_states(k, p, k, p * (1 + 1e-12), thr, 1e-10) <= 2e-12
    with pytest.raises(AssertionError):
        compare_states(k, p, k, p * (1 + 1e-6), thr, 1e-10)
    # an extra zero-mass key on one side: refused unless a neighbouring cell sits within the band of the threshold
    k2 = np.array([[0, 0], [0, 1], [1, 0], [1, 1]], dtype=np.int32)
    p2 = np.array([0.5, 0.3, 0.2, 0.0])
    with pytest.raises(AssertionError):
        compare_states(k2, p2, k, p, thr, 1e-10)
    pb = np.array([0.5, 0.3, thr * (1 + 1e-13)])
    pb2 = np.array([0.5, 0.3, thr * (1 + 1e-13), 0.0])
    compare_states(k2, pb2, k, pb, thr, 1e-10)                       # (1, 0) is in the band and next to (1, 1)
    # ... and never for a key that carries mass, band or not
    with pytest.raises(AssertionError):
        compare_states(k2, np.array([0.5, 0.3, thr * (1 + 1e-13), 1e-9]), k, pb, thr, 1e-10)
    # a far-away band cell does not excuse it
    k3 = np.array([[0, 0], [0, 1], [5, 5]], dtype=np.int32)
    k4 = np.array([[0, 0], [0, 1], [2, 2], [5, 5]], dtype=np.int32)
    with pytest.raises(AssertionError):
        compare_states(k4, np.array([0.5, 0.3, 0.0, thr]), k3, np.array([0.5, 0.3, thr]), thr, 1e-10)
