"""gbees_marginal_noalloc (the one entry point that allocates nothing: scratch in a static device array) against
the existing path gbees_marginal, on two calls in a row. In a file of its own that pytest collects last."""
import numpy as np
import pytest

from paper_2508_13986_b200 import workloads as W

pytestmark = pytest.mark.gpu


def _sorted(keys, p):
    order = np.lexsort(keys.T[::-1])
    return keys[order], p[order]


def test_marginal_noalloc_matches_gbees_marginal_on_two_calls_in_a_row():
    import torch
    from paper_2508_13986_b200 import Gbees, binding
    cfg = W.config2()
    cfg.update(thresh=1e-5, max_cells=1 << 20)
    g = Gbees(cfg["n"], cfg["dx"], cfg["thresh"], cfg["dyn"], cfg["params"], cfl=cfg["cfl"], max_cells=cfg["max_cells"])
    g.init_gaussian(cfg["mean"], cfg["cov"])
    assert g.run(1e300, max_steps=6, prune_every=3) == 6
    N = g.count()
    assert 10_000 < N <= binding.NOALLOC_MAX_CELLS
    # inputs: the exported state in caller-owned device buffers; outputs: caller-owned device buffers
    keys_t = torch.empty((N, cfg["n"]), dtype=torch.int32, device="cuda")
    p_t = torch.empty(N, dtype=torch.float64, device="cuda")
    assert g.export_device(keys_t, p_t) == N
    out_k = torch.empty((N, 3), dtype=torch.int32, device="cuda")
    out_p = torch.empty(N, dtype=torch.float64, device="cuda")
    torch.cuda.synchronize()
    # two calls in a row on the shared scratch array: the second (other dims, fewer cells) must not see the first
    for dims in ([0, 1, 2], [5, 3]):
        m = len(dims)
        ok_view = out_k.view(-1)[: N * m].view(N, m)
        got = binding.marginal_noalloc(keys_t, p_t, dims, ok_view, out_p)
        torch.cuda.synchronize()
        gk, gp = _sorted(ok_view[:got].cpu().numpy(), out_p[:got].cpu().numpy())
        wk, wp = g.marginal(dims)                                  # the existing path (sorted)
        assert got == len(wp)
        assert np.array_equal(gk, wk), f"dims {dims}: marginal key sets differ"
        assert np.max(np.abs(gp - wp)) <= 1e-12 * np.max(np.abs(wp))   # the tolerance of test_marginals_of_the_6d_pdf
        assert gp.sum() == pytest.approx(1.0, abs=1e-12)
    # sizes beyond the static scratch are refused with a clear error, nothing is launched
    big_k = torch.zeros((binding.NOALLOC_MAX_CELLS + 1, cfg["n"]), dtype=torch.int32, device="cuda")
    big_p = torch.zeros(binding.NOALLOC_MAX_CELLS + 1, dtype=torch.float64, device="cuda")
    with pytest.raises(binding.GbeesError) as ei:
        binding.marginal_noalloc(big_k, big_p, [0], out_k, out_p)
    assert ei.value.code == -4 and "GBEES_NOALLOC_MAX_CELLS" in str(ei.value)
    # an output buffer that is too small: GBEES_ERR_BUFFER
    with pytest.raises(binding.GbeesError) as ei:
        binding.marginal_noalloc(keys_t, p_t, [0, 1, 2], out_k[:8], out_p[:8])
    assert ei.value.code == -5
    g.close()
