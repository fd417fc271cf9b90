"""Distribution metrics of the paper's validation (TEST INFRASTRUCTURE ONLY), written as their
definitions with a python dict join:
  BC = sum_i sqrt(P_i P0_i)                     Eq. (9),  PAPER.md:347-352 (P = cell probabilities, sum 1)
  E  = prod(h) sum_i |p_i - p0_i| = sum_i |P_i - P0_i|    PAPER.md:362-366 (p = density, P = p prod(h) = mass)
over the union of the two active sets; a cell missing from one set has probability 0 there."""
import math


def bc_and_l1(keys_a, p_a, keys_b, p_b):
    a = {tuple(k): float(v) for k, v in zip(keys_a.tolist(), p_a.tolist())}
    b = {tuple(k): float(v) for k, v in zip(keys_b.tolist(), p_b.tolist())}
    bc, l1 = 0.0, 0.0
    for k in sorted(set(a) | set(b)):
        pa, pb = a.get(k, 0.0), b.get(k, 0.0)
        if pa > 0.0 and pb > 0.0:
            bc += math.sqrt(pa * pb)
        l1 += abs(pa - pb)
    return bc, l1
