"""BASELINE config 4: hashtable / compaction device code against the numpy oracle, and the probe
counts against the closed forms of PAPER.md:192 (tests/golden/probe_counts.txt)."""
import os

import numpy as np
import pytest

from oracle import ht_oracle
from paper_2508_13986_b200 import workloads as W

GOLD = os.path.join(os.path.dirname(os.path.abspath(__file__)), "golden", "probe_counts.txt")


def golden():
    rows = [ln.split() for ln in open(GOLD) if ln.strip() and not ln.startswith("#")]
    return {float(a): (float(s), float(u)) for a, s, u in rows}


def test_golden_values_are_the_papers_formulas():
    for a, (s, u) in golden().items():
        assert s == pytest.approx(0.5 * (1 + 1 / (1 - a)), rel=1e-12)
        assert u == pytest.approx(0.5 * (1 + 1 / (1 - a) ** 2), rel=1e-12)


@pytest.mark.parametrize("alpha", [0.3, 0.5, 0.7])
def test_P11_oracle_linear_probing_matches_closed_forms(alpha):
    """The literal linear-probing simulation reproduces the closed forms (pins the oracle's probe count)."""
    s, u = ht_oracle.linear_probe_counts(60000, alpha, W.S0 + 41)
    gs, gu = golden()[alpha]
    assert s == pytest.approx(gs, rel=0.04)
    assert u == pytest.approx(gu, rel=0.08)


def test_config4_keys_are_distinct_and_in_range():
    k = W.config4_keys(20000)
    assert len(k) == 20000 and len(np.unique(k)) == 20000
    assert int(k.max()) < (1 << 60)


def test_oracle_lookup_and_compact_definitions():
    keys = np.array([5, 9, 2, 7], dtype=np.uint64)
    assert ht_oracle.lookup_found(keys, np.array([2, 3, 9, 10], dtype=np.uint64)).tolist() == [True, False, True, False]
    assert ht_oracle.compact(keys, np.array([0, 1, 0, 1], dtype=np.uint8)).tolist() == [5, 2]


@pytest.mark.gpu
@pytest.mark.parametrize("alpha", [0.3, 0.5, 0.8])
def test_gpu_table_insert_lookup_compact(alpha):
    import torch
    from paper_2508_13986_b200 import HashTable
    K = 1_000_000
    keys = W.config4_keys(K)
    rng = np.random.default_rng(W.S0 + 42)
    ht = HashTable(int(np.ceil(K / alpha)))
    kt = torch.from_numpy(keys.view(np.int64)).cuda()
    idx = torch.empty(K, dtype=torch.int32, device="cuda")
    probes_ins = ht.insert(kt, idx)
    rows = idx.cpu().numpy().view(np.uint32)
    assert np.array_equal(np.sort(rows), np.arange(K, dtype=np.uint32))          # rows are a permutation of 0..K-1
    # successful lookups return the row assigned at insert; probe counts follow PAPER.md:192
    out = torch.empty(K, dtype=torch.int32, device="cuda")
    probes_hit = ht.lookup(kt, out)
    assert torch.equal(out, idx)
    gs, gu = golden()[alpha]
    assert probes_hit / K == pytest.approx(gs, rel=0.03)
    assert probes_ins / K == pytest.approx(gs, rel=0.03)                             # insert cost == successful search
    # 2n face-neighbour queries of every key (uniform keys: almost all unsuccessful)
    unit = np.uint64(1) << (np.uint64(10) * np.arange(6, dtype=np.uint64))
    sub = keys[:200_000]
    q = np.concatenate([sub + u for u in unit] + [sub - u for u in unit])
    found = ht_oracle.lookup_found(keys, q)
    qt = torch.from_numpy(q.view(np.int64)).cuda()
    qo = torch.empty(len(q), dtype=torch.int32, device="cuda")
    probes_q = ht.lookup(qt, qo)
    got = qo.cpu().numpy().view(np.uint32) != 0xFFFFFFFF
    assert np.array_equal(got, found)
    assert found.mean() < 0.01
    assert probes_q / len(q) == pytest.approx(gu, rel=0.05)
    # cooperative probing (tiles of 4, 8, 32 lanes): same answers, same probe counts
    for width in (4, 8, 32):
        qo2 = torch.empty(len(q), dtype=torch.int32, device="cuda")
        assert ht.lookup_coop(qt, qo2, width) == probes_q and torch.equal(qo2, qo)
        out3 = torch.empty(K, dtype=torch.int32, device="cuda")
        assert ht.lookup_coop(kt, out3, width) == probes_hit and torch.equal(out3, idx)
    # delete 30 %, compact (stable), rebuild
    dele = (rng.random(K) < 0.3).astype(np.uint8)
    dt_ = torch.from_numpy(dele).cuda()
    kept = ht.compact(kt, dt_)
    want = ht_oracle.compact(keys, dele)
    assert kept == len(want)
    assert np.array_equal(kt[:kept].cpu().numpy().view(np.uint64), want)
    out2 = torch.empty(K, dtype=torch.int32, device="cuda")
    ht.lookup(torch.from_numpy(keys.view(np.int64)).cuda(), out2)
    r2 = out2.cpu().numpy().view(np.uint32)
    assert np.array_equal(r2 != 0xFFFFFFFF, dele == 0)                              # deleted keys are gone
    assert np.array_equal(r2[dele == 0], np.arange(kept, dtype=np.uint32))          # survivors: row = new position
    ht.close()
