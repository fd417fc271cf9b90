"""Config-4 oracle (TEST INFRASTRUCTURE ONLY): what a key -> row table must answer, written with
plain numpy set operations, and a literal simulation of open addressing with linear probing
 that counts probes, used to pin the closed forms the paper quotes.
Shares nothing with the CUDA path (own hash: numpy's PCG64 draws the home slots)."""
import numpy as np


def lookup_found(keys, queries):
    """found[i] = queries[i] is one of keys (the definition of a successful lookup)."""
    s = np.sort(np.asarray(keys))
    pos = np.searchsorted(s, queries)
    pos[pos == len(s)] = len(s) - 1
    return s[pos] == queries


def compact(keys, delete):
    """Surviving keys in their original order (stable stream compaction)."""
    return np.asarray(keys)[np.asarray(delete) == 0]


def linear_probe_counts(n_keys, alpha, seed, n_miss=None):
    """Insert n_keys keys with uniformly random home slots into a table of n_keys/alpha slots by
    linear probing; return (mean probes of a successful search, mean probes of an unsuccessful one).
    A probe = one slot inspected, the empty slot that ends an unsuccessful search included."""
    rng = np.random.default_rng(seed)
    m = int(round(n_keys / alpha))
    used = np.zeros(m, dtype=bool)
    home = rng.integers(0, m, n_keys)
    succ = 0
    for h in home.tolist():           # insertion cost == later successful-search cost of that key
        s, p = h, 1
        while used[s]:
            s = s + 1 if s + 1 < m else 0
            p += 1
        used[s] = True
        succ += p
    n_miss = n_miss or n_keys
    miss = 0
    for h in rng.integers(0, m, n_miss).tolist():
        s, p = h, 1
        while used[s]:
            s = s + 1 if s + 1 < m else 0
            p += 1
        miss += p
    return succ / n_keys, miss / n_miss
