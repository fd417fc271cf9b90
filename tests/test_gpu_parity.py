"""GPU-vs-oracle parity through the C ABI (python binding = argument marshalling only)."""
import itertools

import numpy as np
import pytest

from oracle.binding import Oracle
from paper_2508_13986_b200 import workloads as W
from util import compare_states, key_hash, sort_state

pytestmark = pytest.mark.gpu


def G(*a, **k):
    from paper_2508_13986_b200 import Gbees
    return Gbees(*a, **k)


def box(lo, hi):
    return np.array(list(itertools.product(*[range(a, b) for a, b in zip(lo, hi)])), dtype=np.int32)


def pair_raw(n, h, dyn, params, keys, p, origin, hi_res=1, limiter=0, cfl=0.9):
    o = Oracle(n, h, 1e-300, dyn, params, cfl=cfl, hi_res=hi_res, limiter=limiter)
    o.set_flags(grow=False, normalise=False)
    o.import_state(origin, keys, p)
    g = G(n, h, 1e-300, dyn, params, cfl=cfl, hi_res=hi_res, limiter=limiter, no_grow=True, no_normalise=True,
          max_cells=1 << 16)
    g.import_state(origin, keys, p)
    return g, o


@pytest.mark.parametrize("n,axis,sign", [(1, 0, 1), (3, 1, 1), (3, 2, -1), (6, 4, 1), (6, 0, -1)])
def test_courant_one_shift_bit_exact(n, axis, sign):
    rng = np.random.default_rng(W.S0 + 202)
    v = np.zeros(n); v[axis] = 2.0 * sign
    hi = [3] * n; hi[axis] = 12
    keys = box([0] * n, hi)
    p = rng.integers(0, 64, len(keys)).astype(np.float64) * 2.0 ** -9
    p[(keys[:, axis] < 2) | (keys[:, axis] >= 10)] = 0.0
    for hi_res, limiter in [(0, 0), (1, 0), (1, 1)]:
        g, o = pair_raw(n, [0.5] * n, 4, v, keys, p, np.zeros(n), hi_res, limiter, cfl=1.0)
        assert g.step() == o.step() == 0.25
        gk, gp = g.export(); ok, op = o.export()
        assert np.array_equal(gk, ok) and np.array_equal(gp, op)


CASES = [
    (3, 6, 0, [10, 8 / 3, 28], [-11.5, -10, 9.5]),
    (3, 9, 1, [4.0, 1.0, 48.0], [-11.5, -10, 9.5]),
    (4, 5, 2, [4.0], [4.01, 4, 4, 4]),
    (5, 4, 2, [4.0], [4.01, 4, 4, 4, 4]),
    (6, 4, 2, [4.0], [4.01, 4, 4, 4, 4, 4]),
    (6, 3, 3, None, [0.3, -0.2, 0.1, 0.5, -0.4, 0.2]),
    (2, 20, 3, None, [0.3, -0.2]),
    (1, 50, 3, [-0.7], [0.3]),
]


@pytest.mark.parametrize("n,side,dyn,params,origin", CASES)
@pytest.mark.parametrize("ragged", [False, True])
def test_frozen_grid_flux_update(n, side, dyn, params, origin, ragged):
    """a2-a6 on a frozen grid (no grow, no normalise): random masses incl. negatives, ragged sets."""
    rng = np.random.default_rng(W.S0 + 207 + 10 * n + dyn + ragged)
    if params is None:
        params = rng.normal(0, 0.3, (n, n)).ravel()
    h = rng.uniform(0.3, 0.6, n)
    keys = box([-(side // 2)] * n, [side - side // 2] * n)
    if ragged:
        keys = keys[rng.random(len(keys)) < 0.6]
    p = rng.random(len(keys)) - 0.1
    for hi_res, limiter in [(0, 0), (1, 0), (1, 1)]:
        g, o = pair_raw(n, h, dyn, params, keys, p, origin, hi_res, limiter)
        for _ in range(3):
            dg, do = g.step(), o.step()
            assert dg == do                                   # dt bit-identical (A12)
            gk, gp = g.export(); ok, op = o.export()
            assert np.array_equal(gk, ok)
            assert np.max(np.abs(gp - op)) <= 1e-12 * np.max(np.abs(op))
            assert g.last_mass() == pytest.approx(o.last_mass(), rel=1e-12)


def run_lockstep(cfg, steps, check_every=1, rtol_step=1e-10):
    o = Oracle(cfg["n"], cfg["dx"], cfg["thresh"], cfg["dyn"], cfg["params"], cfl=cfg["cfl"])
    g = G(cfg["n"], cfg["dx"], cfg["thresh"], cfg["dyn"], cfg["params"], cfl=cfg["cfl"], max_cells=cfg["max_cells"])
    o.init_gaussian(cfg["mean"], cfg["cov"]); g.init_gaussian(cfg["mean"], cfg["cov"])
    # the two normalisation sums add the N initial masses in different orders: error <= N eps
    compare_states(*g.export(), *o.export(), cfg["thresh"], 1e-11, what="init")
    worst = 0.0
    for k in range(1, steps + 1):
        dg, do = g.step(), o.step()
        assert abs(dg - do) <= 1e-14 * do, f"dt mismatch at step {k}: {dg} vs {do}"
        if cfg["prune_every"] and k % cfg["prune_every"] == 0:
            g.prune(); o.prune()
        if k % check_every == 0 or k == steps:
            assert g.count() == o.count(), f"step {k}: {g.count()} vs {o.count()} cells"
            worst = max(worst, compare_states(*g.export(), *o.export(), cfg["thresh"], rtol_step, what=f"step {k}"))
            assert g.time() == pytest.approx(o.time(), rel=1e-14)
    return worst, g, o


def test_config0_lockstep_20_steps():
    worst, g, o = run_lockstep(W.config0(), 20)
    assert worst <= 1e-10
    assert g.stats()["steps"] == 20


def test_lorenz96_6d_small_lockstep():
    cfg = W.config2()
    cfg.update(thresh=1e-5, max_cells=1 << 20)   # same physics, fewer cells: oracle finishes in seconds
    worst, g, o = run_lockstep(cfg, 7)
    assert worst <= 1e-10


def test_config1_short_with_corrections():
    cfg = W.config1()
    cfg.update(dx=[0.5] * 3)
    o = Oracle(cfg["n"], cfg["dx"], cfg["thresh"], cfg["dyn"], cfg["params"], cfl=cfg["cfl"])
    g = G(cfg["n"], cfg["dx"], cfg["thresh"], cfg["dyn"], cfg["params"], cfl=cfg["cfl"], max_cells=1 << 18)
    o.init_gaussian(cfg["mean"], cfg["cov"]); g.init_gaussian(cfg["mean"], cfg["cov"])
    for tm, z in zip([0.02, 0.04], cfg["z"]):
        k = 0
        while o.time() < tm:
            dg, do = g.step(tm - g.time()), o.step(tm - o.time())
            assert abs(dg - do) <= 1e-14 * do
            g.prune(); o.prune()
            k += 1
        assert g.time() == o.time() == tm
        # measurement near the current blob so the posterior keeps mass on the grid
        kk, pp = o.export()
        zc = np.array(cfg["mean"]) + (pp[:, None] * kk).sum(0) * np.array(cfg["dx"]) + 0.3
        g.correct(zc, cfg["R"]); o.correct(zc, cfg["R"])
        g.prune(); o.prune()
        compare_states(*g.export(), *o.export(), cfg["thresh"], 1e-10, what=f"after correct t={tm}")


def test_errors_and_edges():
    from paper_2508_13986_b200 import GbeesError
    g = G(3, [0.5] * 3, 2e-5, 0, [10, 8 / 3, 28], max_cells=1000)
    with pytest.raises(GbeesError) as e:
        g.init_gaussian([-11.5, -10, 9.5], np.eye(3))   # needs 1357 cells
    assert e.value.code == -4
    g = G(3, [0.5] * 3, 2e-5, 0, [10, 8 / 3, 28], max_cells=4096)
    with pytest.raises(GbeesError) as e:
        g.init_gaussian([0, 0, 0], np.array([[1, 2, 0], [2, 1, 0], [0, 0, 1.0]]))
    assert e.value.code == -3
    with pytest.raises(GbeesError) as e:
        g.step()                                           # empty grid
    assert e.value.code == -6
    with pytest.raises(GbeesError) as e:
        G(3, [0.5] * 3, 0.0, 0, [10, 8 / 3, 28])          # threshold must be positive
    assert e.value.code == -1
    # key range: 6-D fields hold [-512, 511]
    g = G(6, [0.5] * 6, 1e-3, 4, [1.0] * 6, max_cells=4096)
    g.import_state(np.zeros(6), np.array([[511, 0, 0, 0, 0, 0]], dtype=np.int32), np.array([1.0]))
    with pytest.raises(GbeesError) as e:
        g.step()
    assert e.value.code == -7
    # single cell, constant velocity: grows its downwind face/edge neighbours, mass stays 1
    g = G(3, [0.5] * 3, 1e-3, 4, [1.0, -1.0, 0.0], max_cells=4096)
    g.import_state(np.zeros(3), np.zeros((1, 3), dtype=np.int32), np.array([1.0]))
    g.step()
    k, p = g.export()
    assert len(k) == 4 and p.sum() == pytest.approx(1.0, abs=1e-15)


def oracle_run(cfg, t_end=None, steps=None):
    o = Oracle(cfg["n"], cfg["dx"], cfg["thresh"], cfg["dyn"], cfg["params"], cfl=cfg["cfl"])
    o.init_gaussian(cfg["mean"], cfg["cov"])
    k = 0
    while (t_end is None or o.time() < t_end) and (steps is None or k < steps):
        o.step(t_end - o.time() if t_end is not None else 0.0)
        k += 1
        if cfg["prune_every"] and k % cfg["prune_every"] == 0:
            o.prune()
    return o, k


@pytest.mark.parametrize("run_mode", [0, 1])
def test_run_persistent_loop_config0(run_mode):
    """a9: gbees_run (persistent cooperative kernel / host loop) == the oracle's step/prune sequence."""
    cfg = W.config0()
    g = G(cfg["n"], cfg["dx"], cfg["thresh"], cfg["dyn"], cfg["params"], cfl=cfg["cfl"], max_cells=cfg["max_cells"],
          run_mode=run_mode)
    g.init_gaussian(cfg["mean"], cfg["cov"])
    assert g.run(1e300, max_steps=20, prune_every=1) == 20
    o, _ = oracle_run(cfg, steps=20)
    assert g.time() == pytest.approx(o.time(), rel=1e-14)
    assert compare_states(*g.export(), *o.export(), cfg["thresh"], 1e-9, what="cfg0 run") <= 1e-9
    st = g.stats()
    assert st["steps"] == 20 and st["prunes"] == 20


@pytest.mark.parametrize("prune_every", [0, 2, 5])
def test_run_persistent_loop_lorenz96_to_time(prune_every):
    cfg = W.config2()
    cfg.update(thresh=1e-5, max_cells=1 << 20, prune_every=prune_every)
    g = G(cfg["n"], cfg["dx"], cfg["thresh"], cfg["dyn"], cfg["params"], cfl=cfg["cfl"], max_cells=cfg["max_cells"])
    g.init_gaussian(cfg["mean"], cfg["cov"])
    o, k = oracle_run(cfg, t_end=0.05)
    assert g.run(0.05, prune_every=prune_every) == k
    assert g.time() == o.time() == 0.05
    compare_states(*g.export(), *o.export(), cfg["thresh"], 1e-9, what="L96 run")
    # the context stays usable call-by-call after a persistent run (buffers swapped back correctly)
    assert abs(g.step() - o.step()) <= 1e-14
    g.prune(); o.prune()
    compare_states(*g.export(), *o.export(), cfg["thresh"], 1e-9, what="L96 run + step + prune")


@pytest.mark.parametrize("run_mode", [2, 3])
def test_run_modes_graph_and_cooperative_are_observationally_identical(run_mode):
    """a9: gbees_run with the chunks of steps captured as a CUDA graph (run_mode 2) and as
    ONE cooperative launch over the whole GPU with grid barriers between the phases (run_mode 3, the paper's
    execution model) gives the oracle's step / prune sequence, like the default stream of launches."""
    import torch
    cfg = W.config2()
    cfg.update(thresh=1e-5, max_cells=1 << 20)
    stream = torch.cuda.Stream()                                   # (a graph cannot be captured on the legacy default stream)
    g = G(cfg["n"], cfg["dx"], cfg["thresh"], cfg["dyn"], cfg["params"], cfl=cfg["cfl"], max_cells=cfg["max_cells"],
          run_mode=run_mode, stream=stream.cuda_stream)
    g.init_gaussian(cfg["mean"], cfg["cov"])
    o, k = oracle_run(cfg, t_end=0.2)
    assert k > 20                                                   # more than one graph chunk
    assert g.run(0.2, prune_every=cfg["prune_every"]) == k
    assert g.time() == o.time() == 0.2
    compare_states(*g.export(), *o.export(), cfg["thresh"], 1e-9, what=f"run_mode {run_mode}")
    assert g.stats()["steps"] == k and g.stats()["prunes"] == k // cfg["prune_every"]


def test_config2_full_size_against_oracle_golden():
    """BASELINE config 2 at full size, in the launch configuration bench.py times (gbees_run, device-side
    step control): step count, final time, cell counts after every 5th step and the masses of 128
    sampled cells against the oracle's stored result (tests/golden/cfg2_full_oracle.json, written by
    tests/golden/make_cfg2_golden.py, which calls only oracle/)."""
    import json
    import os
    gold = json.load(open(os.path.join(os.path.dirname(os.path.abspath(__file__)), "golden", "cfg2_full_oracle.json")))
    cfg = W.config2()
    g = G(cfg["n"], cfg["dx"], cfg["thresh"], cfg["dyn"], cfg["params"], cfl=cfg["cfl"], max_cells=cfg["max_cells"])
    g.init_gaussian(cfg["mean"], cfg["cov"])
    counts = {0: g.count()}
    done = 0
    while g.time() < cfg["t_end"]:                      # chunks of 5 steps so the cell counts can be compared
        done += g.run(cfg["t_end"], max_steps=5, prune_every=0)
        if done % cfg["prune_every"] == 0:
            g.prune()
        counts[done] = g.count()
    assert done == gold["steps"]
    assert g.time() == gold["t"] == cfg["t_end"]
    for k, cnt in counts.items():
        assert cnt == gold["cells_after_each_step"][k], f"cell count after step {k}"
    gk, gp = g.export()
    assert len(gp) == gold["final_cells"]
    assert gp.sum() == pytest.approx(1.0, abs=1e-12)
    lut = {tuple(k): v for k, v in zip(gk.tolist(), gp.tolist())}
    got = np.array([lut[tuple(k)] for k in gold["sample_keys"]])      # KeyError = active sets differ
    want = np.array(gold["sample_p"])
    assert np.max(np.abs(got - want)) <= 1e-8 * gold["p_max"]
    # and the same job through one gbees_run call gives the same state
    g2 = G(cfg["n"], cfg["dx"], cfg["thresh"], cfg["dyn"], cfg["params"], cfl=cfg["cfl"], max_cells=cfg["max_cells"])
    g2.init_gaussian(cfg["mean"], cfg["cov"])
    assert g2.run(cfg["t_end"], prune_every=cfg["prune_every"]) == gold["steps"]
    k2, p2 = g2.export()
    assert np.array_equal(k2, gk) and np.max(np.abs(p2 - gp)) <= 1e-12 * gp.max()


def test_config2_full_size_every_cell_against_the_live_oracle():
    """BASELINE config 2 (the headline) at full size, element by element (north_star: identical active cell
    sets, probabilities within 1e-10 per step / 1e-8 after the run; compare every 10th step +
    final). The oracle runs live beside the GPU (about 4.5 minutes on one host core); the GPU goes through
    gbees_run with device-side step control and prune_every = 5, the launch configuration bench.py times."""
    cfg = W.config2()
    o = Oracle(cfg["n"], cfg["dx"], cfg["thresh"], cfg["dyn"], cfg["params"], cfl=cfg["cfl"])
    g = G(cfg["n"], cfg["dx"], cfg["thresh"], cfg["dyn"], cfg["params"], cfl=cfg["cfl"], max_cells=cfg["max_cells"])
    o.init_gaussian(cfg["mean"], cfg["cov"]); g.init_gaussian(cfg["mean"], cfg["cov"])
    k, worst = 0, 0.0
    while o.time() < cfg["t_end"]:
        k0 = k
        while k < k0 + 10 and o.time() < cfg["t_end"]:
            o.step(cfg["t_end"] - o.time()); k += 1
            if k % cfg["prune_every"] == 0:
                o.prune()
        assert g.run(cfg["t_end"], max_steps=10, prune_every=cfg["prune_every"]) == k - k0
        assert g.time() == o.time()                          # dt bit-identical step after step (A12)
        gk, gp = sort_state(*g.export(sort=False)); ok, op = sort_state(*o.export(sort=False))
        assert np.array_equal(gk, ok), f"step {k}: active sets differ ({len(gk)} vs {len(ok)} cells)"
        err = np.max(np.abs(gp - op)) / np.max(np.abs(op))
        worst = max(worst, err)
        assert err <= 1e-10 * k, f"step {k}: max-norm relative error {err:.3e}"   # 1e-10 per step, compounded
    assert k == 105 and len(gp) == 877679
    assert worst <= 1e-8
    assert gp.sum() == pytest.approx(1.0, abs=1e-12)


def test_config3_tenth_scale_full_run_against_oracle_golden():
    """The 1/10-scale twin of BASELINE config 3 (dx = 0.5, 6 M -> 10 M cells, all 50 steps, prune every 5;
    SURVEY.md 8(d)) against the oracle's stored result (tests/golden/cfg3s_full_oracle.json, written by
    tests/golden/make_cfg3s_golden.py, which calls only oracle/ and takes hours): after EVERY prune the cell
    count and the sha256 of the sorted int32 key array (bit-exact active sets); at the end 4096 sampled
    masses (1e-8), the six 1-D marginals and the first two moments. A golden file from an interrupted
    generator run holds fewer prunes: whatever it holds is compared."""
    import json
    import os
    path = os.path.join(os.path.dirname(os.path.abspath(__file__)), "golden", "cfg3s_full_oracle.json")
    if not os.path.exists(path):
        pytest.skip("tests/golden/cfg3s_full_oracle.json has not been generated")
    gold = json.load(open(path))
    cfg = W.config3(dx=0.5)
    g = G(cfg["n"], cfg["dx"], cfg["thresh"], cfg["dyn"], cfg["params"], cfl=cfg["cfl"], max_cells=1 << 25)
    g.init_gaussian(cfg["mean"], cfg["cov"])
    assert g.count() == gold["cells_initial"]
    done = 0
    for k in sorted(int(x) for x in gold["after_prune"]):
        assert g.run(1e300, max_steps=k - done, prune_every=cfg["prune_every"]) == k - done
        done = k
        want = gold["after_prune"][str(k)]
        assert g.count() == want["cells"], f"cell count after the prune at step {k}"
        assert g.time() == pytest.approx(want["t"], rel=1e-13)
        ks, ps = sort_state(*g.export(sort=False))
        assert key_hash(ks) == want["keys_sha256"], f"active set after the prune at step {k}"
        assert ps.max() == pytest.approx(want["p_max"], rel=1e-8)
    assert done >= 5
    if "final" in gold:
        f = gold["final"]
        assert done == f["steps"] == cfg["steps"] and len(ps) == f["cells"]
        # sampled masses: the sample keys are looked up in the sorted GPU state through the packed sort key
        sk = np.asarray(f["sample_keys"], dtype=np.int32)
        pack = lambda a: sum((a[:, j].astype(np.int64) + 512) << (10 * (5 - j)) for j in range(6))
        pos = np.searchsorted(pack(ks), pack(sk))
        assert np.array_equal(ks[pos], sk)                   # every sampled key is active
        assert np.max(np.abs(ps[pos] - np.asarray(f["sample_p"]))) <= 1e-8 * f["p_max"]
        x = ks.astype(np.float64)
        mean = ps @ x
        d = x - mean
        assert np.allclose(mean, f["mean_index_units"], rtol=0, atol=1e-8)
        assert np.allclose(d.T @ (d * ps[:, None]), f["cov_index_units"], rtol=1e-8, atol=1e-8)
        for j, mg in enumerate(f["marginals_1d"]):
            u, inv = np.unique(ks[:, j], return_inverse=True)
            assert u.tolist() == mg["coords"]
            assert np.allclose(np.bincount(inv, weights=ps), mg["mass"], rtol=0, atol=1e-10)


def test_config1_full_run_with_corrections_bench_sequence():
    """BASELINE config 1 at full size through the call sequence bench.py times (gbees_run to each
    measurement time, correct, prune): final state within 1e-8 (north_star) of the oracle's."""
    cfg = W.config1()
    g = G(cfg["n"], cfg["dx"], cfg["thresh"], cfg["dyn"], cfg["params"], cfl=cfg["cfl"], max_cells=cfg["max_cells"])
    o = Oracle(cfg["n"], cfg["dx"], cfg["thresh"], cfg["dyn"], cfg["params"], cfl=cfg["cfl"])
    g.init_gaussian(cfg["mean"], cfg["cov"]); o.init_gaussian(cfg["mean"], cfg["cov"])
    assert g.count() == o.count() == 4067                       # initial set of cfg1
    total = 0
    for tm, z in zip(cfg["t_meas"], cfg["z"]):
        k = 0
        while o.time() < tm:
            o.step(tm - o.time()); k += 1
            if k % cfg["prune_every"] == 0:
                o.prune()
        assert g.run(tm, prune_every=cfg["prune_every"]) == k
        total += k
        assert g.time() == o.time() == tm
        compare_states(*g.export(), *o.export(), cfg["thresh"], 1e-8, what=f"before the correction at t={tm}")
        g.correct(z, cfg["R"]); o.correct(z, cfg["R"])
        g.prune(); o.prune()
        compare_states(*g.export(), *o.export(), cfg["thresh"], 1e-8, what=f"after the correction at t={tm}")
    assert g.stats()["steps"] == total


def test_linear_6d_stress_twin_lockstep():
    """BASELINE config 3's dynamics and recipe on a coarse grid (dx = 1.0; the oracle finishes in seconds)."""
    cfg = W.config3(dx=1.0)
    cfg.update(thresh=1e-8, max_cells=1 << 21)
    worst, g, o = run_lockstep(cfg, 10)
    assert worst <= 1e-10
    assert g.stats()["prunes"] == 2


def test_export_buffer_contract_and_device_export():
    import torch
    from paper_2508_13986_b200 import GbeesError
    from paper_2508_13986_b200.binding import lib
    import ctypes as C
    cfg = W.config0()
    g = G(cfg["n"], cfg["dx"], cfg["thresh"], cfg["dyn"], cfg["params"], cfl=cfg["cfl"], max_cells=cfg["max_cells"])
    g.init_gaussian(cfg["mean"], cfg["cov"])
    N = g.count()
    cnt = C.c_int64()
    assert lib().gbees_export(g._h, None, None, 0, C.byref(cnt)) == 0 and cnt.value == N      # count only
    small = np.empty((10, 3), dtype=np.int32); sp = np.empty(10)
    assert lib().gbees_export(g._h, small.ctypes.data, sp.ctypes.data, 10, C.byref(cnt)) == -5     # GBEES_ERR_BUFFER
    assert cnt.value == N
    kd = torch.empty((N + 5, 3), dtype=torch.int32, device="cuda"); pd = torch.empty(N + 5, dtype=torch.float64, device="cuda")
    assert g.export_device(kd, pd) == N
    hk, hp = g.export()
    order = np.lexsort(kd[:N].cpu().numpy().T[::-1])
    assert np.array_equal(kd[:N].cpu().numpy()[order], hk) and np.array_equal(pd[:N].cpu().numpy()[order], hp)
    assert len(set(map(tuple, hk.tolist()))) == N                   # no key twice (store <-> table bijection)
    # a threshold above every cell mass after a step: prune removes everything -> GBEES_ERR_DEGENERATE
    g2 = G(3, [0.5] * 3, 0.9, 4, [1.0, 0.0, 0.0], max_cells=4096)
    g2.import_state(np.zeros(3), np.array([[0, 0, 0], [1, 0, 0]], dtype=np.int32), np.array([0.5, 0.5]))
    with pytest.raises(GbeesError) as e:
        g2.prune()
    assert e.value.code == -6


def test_correct_linear_partial_state_parity():
    """f2: Eq. (4) with y = H x + v on the GPU against the oracle (single-state and 2 x 3 measurement)."""
    cfg = W.config0()
    for H, y, R in [(np.array([[0.0, 0.0, 1.0]]), np.array([9.1]), np.array([[1.0]])),
                    (np.array([[1.0, 0.0, 0.5], [0.0, 2.0, -1.0]]), np.array([-6.9, -29.2]), np.array([[0.9, 0.2], [0.2, 1.4]]))]:
        g = G(cfg["n"], cfg["dx"], cfg["thresh"], cfg["dyn"], cfg["params"], cfl=cfg["cfl"], max_cells=cfg["max_cells"])
        o = Oracle(cfg["n"], cfg["dx"], cfg["thresh"], cfg["dyn"], cfg["params"], cfl=cfg["cfl"])
        g.init_gaussian(cfg["mean"], cfg["cov"]); o.init_gaussian(cfg["mean"], cfg["cov"])
        for _ in range(3):
            g.step(); o.step(); g.prune(); o.prune()
        g.correct_linear(H, y, R); o.correct_linear(H, y, R)
        compare_states(*g.export(), *o.export(), cfg["thresh"], 1e-10, what="after correct_linear")
        g.prune(); o.prune()
        g.step(); o.step()
        compare_states(*g.export(), *o.export(), cfg["thresh"], 1e-10, what="correct_linear + prune + step")


def test_correct_range_nonlinear_measurement_parity():
    """f2, non-linear h(x) = ||x - s||: GPU against the oracle, then a prune and a step."""
    cfg = W.config0()
    g = G(cfg["n"], cfg["dx"], cfg["thresh"], cfg["dyn"], cfg["params"], cfl=cfg["cfl"], max_cells=cfg["max_cells"])
    o = Oracle(cfg["n"], cfg["dx"], cfg["thresh"], cfg["dyn"], cfg["params"], cfl=cfg["cfl"])
    g.init_gaussian(cfg["mean"], cfg["cov"]); o.init_gaussian(cfg["mean"], cfg["cov"])
    for _ in range(2):
        g.step(); o.step(); g.prune(); o.prune()
    s0 = np.array([-9.0, -8.5, 12.0])
    g.correct_range(s0, 3.0, 0.5); o.correct_range(s0, 3.0, 0.5)
    compare_states(*g.export(), *o.export(), cfg["thresh"], 1e-10, what="after correct_range")
    g.prune(); o.prune(); g.step(); o.step()
    compare_states(*g.export(), *o.export(), cfg["thresh"], 1e-10, what="correct_range + prune + step")


def test_paper_lorenz63_scenario_soft_sanity():
    """The paper's own Lorenz '63 run: z-shifted form with (sigma, b, r) = (4, 1, 48),
    h = 0.5, dt = 1.0 x CFL, t in [0, 2], one measurement y = x3 = -8 (sigma_y = 1) at t = 1. GPU == oracle
    at 1e-8; SOFT comparison with Table 2 (~960 steps, ~24 k cells at most): the
    paper's threshold is not stated, so only the order of magnitude is asserted."""
    par, mean, dx, thr = [4.0, 1.0, 48.0], [-11.5, -10.0, 9.5], [0.5] * 3, 2e-5
    g = G(3, dx, thr, W.DYN_L63_PAPER, par, cfl=1.0, max_cells=1 << 20)
    o = Oracle(3, dx, thr, W.DYN_L63_PAPER, par, cfl=1.0)
    g.init_gaussian(mean, np.eye(3)); o.init_gaussian(mean, np.eye(3))
    steps, max_cells = 0, o.count()
    for leg, t_end in enumerate([1.0, 2.0]):
        k = 0
        while o.time() < t_end:
            o.step(t_end - o.time()); o.prune(); k += 1
            max_cells = max(max_cells, o.count())
        assert g.run(t_end, prune_every=1) == k
        steps += k
        assert g.time() == o.time() == t_end
        compare_states(*g.export(), *o.export(), thr, 1e-8, what=f"paper L63 scenario, t = {t_end}")
        if leg == 0:
            H, y, R = np.array([[0.0, 0.0, 1.0]]), np.array([-8.0]), np.array([[1.0]])
            g.correct_linear(H, y, R); o.correct_linear(H, y, R)
            g.prune(); o.prune()
            compare_states(*g.export(), *o.export(), thr, 1e-8, what="after the measurement at t = 1")
    print(f"paper L63 scenario: {steps} steps (paper ~960), max {max_cells} cells (paper ~24 k)")
    assert 300 <= steps <= 3000 and 2_000 <= max_cells <= 240_000


def test_compare_metrics_and_temporal_convergence():
    """f1: BC (Eq. 9) and the 1-norm E between two GPU runs on the same grid against
    the metrics oracle applied to the ORACLE's states of the same two runs; and the paper's
    temporal-convergence protocol: E against a reference run with a very small
    epsilon decreases with epsilon."""
    from oracle import metrics_oracle as M
    cfg = W.config0()

    def run_gpu(cfl):
        g = G(cfg["n"], cfg["dx"], cfg["thresh"], cfg["dyn"], cfg["params"], cfl=cfl, max_cells=1 << 18)
        g.init_gaussian(cfg["mean"], cfg["cov"])
        g.run(0.05, prune_every=1)
        assert g.time() == 0.05
        return g

    def run_oracle(cfl):
        o = Oracle(cfg["n"], cfg["dx"], cfg["thresh"], cfg["dyn"], cfg["params"], cfl=cfl)
        o.init_gaussian(cfg["mean"], cfg["cov"])
        while o.time() < 0.05:
            o.step(0.05 - o.time()); o.prune()
        return o.export()

    ref = run_gpu(0.02)
    ork, orp = run_oracle(0.02)
    errs = []
    for eps in (1.0, 0.5, 0.2):
        g = run_gpu(eps)
        bc, l1 = g.compare(ref)
        obc, ol1 = M.bc_and_l1(*run_oracle(eps), ork, orp)
        # the states agree to 1e-8 (north_star), so the metrics do
        assert bc == pytest.approx(obc, abs=1e-8) and l1 == pytest.approx(ol1, abs=1e-8)
        bc2, l12 = ref.compare(g)                                   # symmetric
        assert bc2 == pytest.approx(bc, rel=1e-12) and l12 == pytest.approx(l1, rel=1e-10, abs=1e-13)
        assert 0.9 < bc <= 1.0 + 1e-4
        errs.append(l1)
    assert errs[0] > errs[1] > errs[2] > 0.0
    # a run against itself: E = 0; BC = sum of the positive masses = 1 + |negative mass| (A5: negatives are kept)
    bc, l1 = ref.compare(ref)
    assert l1 == 0.0 and bc == pytest.approx(orp[orp > 0].sum(), abs=1e-8) and abs(bc - 1.0) < 1e-4
    print("temporal convergence, E(eps = 1, 0.5, 0.2) vs eps = 0.02:", errs)


def test_resample_parity_and_spatial_convergence():
    """f1, spatial half: runs with cell width eta * h*, eta = 1.25, 1, 0.8, 0.6, against the
    eta = 0.5 reference at C = 0.1. The reference is remapped conservatively onto each coarser grid
    (gbees_resample, reading A19), imported into a context of that spacing and compared with gbees_compare.
    Checked: the remap against oracle/resample_oracle.py cell by cell (same key set, masses 1e-12), mass
    preserved; BC and E against the metrics oracle applied to the ORACLE's runs; E falls and BC rises as
    eta falls."""
    from oracle import metrics_oracle as M, resample_oracle as RO
    cfg = W.config0()
    hstar, t_end, n = 0.5, 0.02, 3
    mean = np.asarray(cfg["mean"], dtype=np.float64)

    def setup(eta):
        dx = [eta * hstar] * n
        thr = cfg["thresh"] * eta ** n                              # the same density threshold on every grid
        return dx, thr

    def run_gpu(eta):
        dx, thr = setup(eta)
        g = G(n, dx, thr, cfg["dyn"], cfg["params"], cfl=0.1, max_cells=1 << 19)
        g.init_gaussian(mean, cfg["cov"])
        g.run(t_end, prune_every=1)
        assert g.time() == t_end
        return g

    def run_oracle(eta):
        dx, thr = setup(eta)
        o = Oracle(n, dx, thr, cfg["dyn"], cfg["params"], cfl=0.1)
        o.init_gaussian(mean, cfg["cov"])
        while o.time() < t_end:
            o.step(t_end - o.time()); o.prune()
        return o.export()

    ref = run_gpu(0.5)
    rk, rp = ref.export()
    ork, orp = run_oracle(0.5)
    assert np.array_equal(rk, ork)
    errs, bcs = [], []
    for eta in (1.25, 1.0, 0.8, 0.6):
        dx, thr = setup(eta)
        # the remap itself: GPU on the GPU's reference state vs the oracle remap of the same state
        gk, gp = ref.resample(mean, dx)
        wk, wp = RO.resample(rk, rp, mean, [0.5 * hstar] * n, mean, dx)
        assert np.array_equal(gk, wk), f"eta {eta}: remapped key sets differ"
        assert np.max(np.abs(gp - wp)) <= 1e-12 * np.max(np.abs(wp))
        assert gp.sum() == pytest.approx(rp.sum(), rel=1e-12)        # mass preserved
        # metrics on the coarse grid
        g = run_gpu(eta)
        tmp = G(n, dx, thr, cfg["dyn"], cfg["params"], cfl=0.1, max_cells=1 << 19)
        tmp.import_state(mean, gk, gp)
        bc, l1 = g.compare(tmp)
        ok2, op2 = run_oracle(eta)
        obc, ol1 = M.bc_and_l1(ok2, op2, *RO.resample(ork, orp, mean, [0.5 * hstar] * n, mean, dx))
        assert bc == pytest.approx(obc, abs=1e-8) and l1 == pytest.approx(ol1, abs=1e-8)
        errs.append(l1); bcs.append(bc)
        tmp.close(); g.close()
    assert errs[0] > errs[1] > errs[2] > errs[3] > 0.0               # E(eta) falls with the cell width
    assert bcs[0] < bcs[1] < bcs[2] < bcs[3] <= 1.0 + 1e-6
    # argument checks: a finer target grid is refused; the same grid is the identity
    with pytest.raises(Exception):
        ref.resample(mean, [0.1] * n)
    ik, ip = ref.resample(mean, [0.5 * hstar] * n)
    assert np.array_equal(ik, rk) and np.allclose(ip, rp, rtol=1e-14, atol=0)
    print("spatial convergence, E(eta = 1.25, 1, 0.8, 0.6) vs eta = 0.5:", errs, "BC:", bcs)


def test_caller_provided_device_arena():
    """every fixed-capacity device structure is carved from a caller-owned torch tensor
    (opts.arena) instead of cudaMalloc; same results; an arena that is too small is refused."""
    import torch
    from paper_2508_13986_b200 import binding
    cfg = W.config2()
    cfg.update(thresh=1e-5, max_cells=1 << 20)
    need = binding.arena_bytes(cfg["n"], cfg["max_cells"])
    arena = torch.empty(need, dtype=torch.uint8, device="cuda")
    free0 = torch.cuda.mem_get_info()[0]
    ga = G(cfg["n"], cfg["dx"], cfg["thresh"], cfg["dyn"], cfg["params"], cfl=cfg["cfl"], max_cells=cfg["max_cells"], arena=arena)
    assert free0 - torch.cuda.mem_get_info()[0] < (8 << 20)         # nothing of that size was allocated behind our back
    gm = G(cfg["n"], cfg["dx"], cfg["thresh"], cfg["dyn"], cfg["params"], cfl=cfg["cfl"], max_cells=cfg["max_cells"])
    for g in (ga, gm):
        g.init_gaussian(cfg["mean"], cfg["cov"])
        assert g.run(1e300, max_steps=7, prune_every=3) == 7
    ka, pa = ga.export(); km, pm = gm.export()
    assert np.array_equal(ka, km) and np.max(np.abs(pa - pm)) <= 1e-12 * pm.max()
    ga.close(); gm.close()
    with pytest.raises(binding.GbeesError) as ei:
        G(cfg["n"], cfg["dx"], cfg["thresh"], cfg["dyn"], cfg["params"], max_cells=cfg["max_cells"], arena=arena[: need // 2])
    assert ei.value.code == -4


def test_marginals_of_the_6d_pdf():
    """f3: the two 3-D marginals of the 6-D Lorenz '96 PDF (and a 1-D, a 2-D one with
    permuted dimensions) by device hash-accumulation against the numpy group-by of the exported state."""
    import ctypes as C
    from oracle import marginal_oracle as MO
    from paper_2508_13986_b200.binding import lib
    cfg = W.config2()
    cfg.update(thresh=1e-5, max_cells=1 << 20)
    g = G(cfg["n"], cfg["dx"], cfg["thresh"], cfg["dyn"], cfg["params"], cfl=cfg["cfl"], max_cells=cfg["max_cells"])
    g.init_gaussian(cfg["mean"], cfg["cov"])
    g.run(1e300, max_steps=6, prune_every=5)
    o, _ = oracle_run(cfg, steps=6)
    keys, p = o.export()                               # the oracle's state: the expected marginals come from it
    for dims in ([0, 1, 2], [3, 4, 5], [4], [5, 0], [0, 1, 2, 3, 4, 5]):
        mk, mp = g.marginal(dims)
        ok, op = MO.marginal(keys, p, dims)
        assert np.array_equal(mk, ok), dims
        assert np.max(np.abs(mp - op)) <= 1e-10 * op.max()
        assert mp.sum() == pytest.approx(1.0, abs=1e-12)
    # buffer contract: count only, too small a buffer
    d = (C.c_int * 3)(0, 1, 2)
    cnt = C.c_int64()
    assert lib().gbees_marginal(g._h, d, 3, None, None, 0, C.byref(cnt)) == 0 and cnt.value == len(MO.marginal(keys, p, [0, 1, 2])[1])
    small = np.empty((4, 3), dtype=np.int32); sp = np.empty(4)
    assert lib().gbees_marginal(g._h, d, 3, small.ctypes.data, sp.ctypes.data, 4, C.byref(cnt)) == -5
    bad = (C.c_int * 2)(1, 1)
    assert lib().gbees_marginal(g._h, bad, 2, None, None, 0, C.byref(cnt)) == -1


def test_config3_midscale_full_run_against_oracle_golden():
    """BASELINE config 3's recipe (linear 6-D f = Ax, 50 steps, prune every 5) on a mid-scale grid
    (dx = 0.7, ~2 M cells: the largest the serial oracle finishes in tens of minutes) through gbees_run,
    against the oracle's stored result (tests/golden/cfg3m_full_oracle.json, written by
    tests/golden/make_cfg3m_golden.py, which calls only oracle/)."""
    import json
    import os
    gold = json.load(open(os.path.join(os.path.dirname(os.path.abspath(__file__)), "golden", "cfg3m_full_oracle.json")))
    cfg = W.config3(dx=0.7)
    g = G(cfg["n"], cfg["dx"], cfg["thresh"], cfg["dyn"], cfg["params"], cfl=cfg["cfl"], max_cells=1 << 24)
    g.init_gaussian(cfg["mean"], cfg["cov"])
    assert g.count() == gold["cells_after_each_step"][0]
    for k in range(5, cfg["steps"] + 1, 5):
        assert g.run(1e300, max_steps=5, prune_every=0) == 5
        g.prune()
        assert g.count() == gold["cells_after_each_step"][k], f"cell count after step {k}"
    assert g.stats()["steps"] == gold["steps"] == cfg["steps"]
    assert g.time() == pytest.approx(gold["t"], rel=1e-13)
    gk, gp = g.export()
    assert len(gp) == gold["final_cells"]
    lut = {tuple(k): v for k, v in zip(gk.tolist(), gp.tolist())}
    got = np.array([lut[tuple(k)] for k in gold["sample_keys"]])      # KeyError = active sets differ
    assert np.max(np.abs(got - np.array(gold["sample_p"]))) <= 1e-8 * gold["p_max"]


def test_config3_tenth_scale_properties_at_full_size():
    """BASELINE config 3 at 1/10 scale (6-10 M cells; the oracle needs ~5 min per step there, so no
    element-wise oracle comparison): properties that hold at any size. (1) through gbees_run, the launch
    configuration bench.py times: masses sum to 1, no key twice, count == stats. (2) P13 reflection
    symmetry at scale: the problem mirrored in axis 0 (A -> D A D, D = diag(-1, 1, ..., 1); N(0, I) is
    symmetric) gives the mirrored key set and the same masses. Eq. (8) as printed looks at LOWER faces
    only, so the CFL step itself is not mirror-symmetric: both runs take the same capped dt."""
    cfg = W.config3(dx=0.5)
    A = np.array(cfg["params"]).reshape(6, 6)
    D = np.diag([-1.0, 1, 1, 1, 1, 1])

    def make(params):
        g = G(cfg["n"], cfg["dx"], cfg["thresh"], cfg["dyn"], params, cfl=cfg["cfl"], max_cells=1 << 25)
        g.init_gaussian(cfg["mean"], cfg["cov"])
        return g

    g = make(A.ravel())
    assert g.run(1e300, max_steps=10, prune_every=5) == 10
    k0, p0 = g.export()
    st = g.stats()
    assert st["n_cells"] == len(p0) > 6_000_000 and st["prunes"] == 2
    assert p0.sum() == pytest.approx(1.0, abs=1e-11)
    assert not np.any(np.all(k0[1:] == k0[:-1], axis=1))            # sorted export: equal neighbours = duplicate key
    cap = 0.7 * st["dt"]
    g.close()

    def capped(params):
        g = make(params)
        for k in range(1, 7):
            assert g.step(cap) == cap
            if k % 3 == 0:
                g.prune()
        out = g.export()
        g.close()
        return out

    k1, p1 = capped(A.ravel())
    k2, p2 = capped((D @ A @ D).ravel())
    k2m = k2.copy(); k2m[:, 0] = -k2m[:, 0]
    order = np.lexsort(k2m.T[::-1])
    assert np.array_equal(k2m[order], k1)
    assert np.max(np.abs(p2[order] - p1)) <= 1e-10 * p1.max()


@pytest.mark.parametrize("prune_every,max_steps", [(3, 17), (0, 9)])
def test_small_grid_persistent_loop_prune_cadence(prune_every, max_steps):
    """a9 on a small grid (single-cluster persistent loop): prune cadences other than 1 and a step limit
    that is not a multiple of the cadence, against the oracle's step / prune sequence; then the context
    keeps working call by call."""
    cfg = W.config0()
    cfg.update(prune_every=prune_every)
    g = G(cfg["n"], cfg["dx"], cfg["thresh"], cfg["dyn"], cfg["params"], cfl=cfg["cfl"], max_cells=cfg["max_cells"])
    g.init_gaussian(cfg["mean"], cfg["cov"])
    assert g.run(1e300, max_steps=max_steps, prune_every=prune_every) == max_steps
    o, _ = oracle_run(cfg, steps=max_steps)
    assert g.time() == pytest.approx(o.time(), rel=1e-14)
    compare_states(*g.export(), *o.export(), cfg["thresh"], 1e-9, what="small-grid run")
    assert g.stats()["launches"] < 40                                  # one launch for the loop, not 4 per step
    assert abs(g.step() - o.step()) <= 1e-14
    g.prune(); o.prune()
    compare_states(*g.export(), *o.export(), cfg["thresh"], 1e-9, what="small-grid run + step + prune")


def test_repeatability_of_the_full_cfg2_run():
    """The paper notes that CUDA's execution order is not deterministic and that the effect on the PDF is
    minimal. Here row allocation (atomicAdd) is the only order-dependent step; it changes
    the order of the mass-sum partials only. Five full cfg2 runs: identical key sets, masses within 1e-12.
    (Stands in for the race detector: compute-sanitizer is closed on this GPU pool.)"""
    cfg = W.config2()
    ref = None
    for rep in range(5):
        g = G(cfg["n"], cfg["dx"], cfg["thresh"], cfg["dyn"], cfg["params"], cfl=cfg["cfl"], max_cells=cfg["max_cells"])
        g.init_gaussian(cfg["mean"], cfg["cov"])
        g.run(cfg["t_end"], prune_every=cfg["prune_every"])
        k, p = g.export()
        g.close()
        if ref is None:
            ref = (k, p)
        else:
            assert np.array_equal(k, ref[0])
            assert np.max(np.abs(p - ref[1])) <= 1e-12 * ref[1].max()
