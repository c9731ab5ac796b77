"""GPU parity of the divergence statistic (``-m gpu``): sparrow_acceptance against the fp64 oracle
on the same synthetic top-20 lists -- alpha element by element, bin counts exactly, the per-bin 5-percentile within
the fp32 evaluation error of alpha (the k-th smallest of perturbed values moves by at most the perturbation)."""
import numpy as np
import pytest
import torch

import oracle
from paper_2606_08446_b200 import workloads as W

pytestmark = pytest.mark.gpu
DEV = "cuda"
TOL = 2e-6


def _run(inp, top_n, bin_tokens, n_bins, quantile):
    from paper_2606_08446_b200 import binding as B
    n_pos = int(inp["positions"].numel())
    alpha = torch.full((max(n_pos, 1),), -1.0, dtype=torch.float32, device=DEV)
    bq = torch.zeros((n_bins,), dtype=torch.float32, device=DEV)
    bc = torch.full((n_bins,), -1, dtype=torch.int32, device=DEV)
    ws = torch.zeros((B.sparrow_acceptance_workspace_bytes(n_bins),), dtype=torch.uint8, device=DEV)
    for _ in range(2):                       # twice: the workspace must be restored by the call
        B.sparrow_acceptance(inp["ids_p"], inp["logp_p"], inp["ids_q"], inp["logp_q"], inp["positions"], top_n, bin_tokens, n_bins,
                             quantile, alpha, bq, bc, ws)
    torch.cuda.synchronize()
    assert B.sparrow_last_launch_count() == (7 if n_pos else 6)
    return alpha[:n_pos].cpu().numpy(), bq.cpu().numpy(), bc.cpu().numpy()


@pytest.mark.parametrize("n_traj,max_len,top_n,bins", [(24, 9000, 20, 6), (3, 700, 20, 19), (40, 3000, 32, 2), (5, 100, 1, 3), (7, 500, 18, 4), (9, 300, 27, 2)])
def test_acceptance_matches_oracle(n_traj, max_len, top_n, bins):
    inp = W.make_acceptance_inputs(n_traj, max_len, top_n=top_n, seed=n_traj, device=DEV)
    a, bq, bc = _run(inp, top_n, 2048, bins, 0.05)
    h = {k: v.cpu().numpy() for k, v in inp.items() if k != "lens"}
    want = oracle.acceptance_rate(h["ids_p"], h["logp_p"].astype(np.float64), h["ids_q"], h["logp_q"].astype(np.float64))
    assert np.abs(a - want).max() <= TOL
    counts, qv = oracle.binned_quantile(want, h["positions"], 2048, bins, float(np.float32(0.05)))
    assert bc.tolist() == counts.tolist()
    for b in range(bins):
        if counts[b] == 0:
            assert np.isnan(bq[b])
        else:
            assert abs(bq[b] - qv[b]) <= TOL, (b, bq[b], qv[b])
    # the statistic the paper tracks decays with length on this workload
    if bins == 6:
        assert bq[0] > bq[3] > 0


def test_acceptance_with_lists_that_are_not_16_byte_aligned():
    """The alpha kernel stages its lists with 16-byte loads only when top_n is a multiple of 4 AND the four arrays are 16-byte
    aligned; copies that start 4 bytes into an allocation must take the scalar path and give the same values."""
    def shifted(t):                          # same values, base pointer + one element (4 bytes)
        buf = torch.empty((t.numel() + 1,), dtype=t.dtype, device=t.device)
        v = buf[1:].view(t.shape)
        v.copy_(t)
        assert v.data_ptr() % 16 != 0 and v.is_contiguous()
        return v
    inp = W.make_acceptance_inputs(6, 400, top_n=20, seed=5, device=DEV)
    ref, _, _ = _run(inp, 20, 2048, 2, 0.05)
    mis = {k: (shifted(v) if k in ("ids_p", "logp_p", "ids_q", "logp_q") else v) for k, v in inp.items()}
    got, _, _ = _run(mis, 20, 2048, 2, 0.05)
    h = {k: v.cpu().numpy() for k, v in inp.items() if k != "lens"}
    want = oracle.acceptance_rate(h["ids_p"], h["logp_p"].astype(np.float64), h["ids_q"], h["logp_q"].astype(np.float64))
    assert np.abs(got - want).max() <= TOL and np.abs(ref - want).max() <= TOL
    assert np.array_equal(got, ref)          # same arithmetic either way, only the staging differs


def test_acceptance_exact_rank_on_the_gpu_values_and_edge_cases():
    """Selection is exact: the reported quantile is bit-for-bit the rank-ceil(q n) element of the GPU's own alphas."""
    from paper_2606_08446_b200 import binding as B
    inp = W.make_acceptance_inputs(16, 5000, seed=7, device=DEV)
    for quantile in (0.05, 0.5, 1.0, 1e-6):
        a, bq, bc = _run(inp, 20, 1024, 5, quantile)
        pos = inp["positions"].cpu().numpy()
        for b in range(5):
            v = np.sort(a[np.minimum(pos // 1024, 4) == b])
            k = max(1, int(np.ceil(float(np.float32(quantile)) * len(v))))
            assert bq[b] == v[k - 1]
    empty = {k: v[:0].contiguous() for k, v in inp.items() if k != "lens"}
    a, bq, bc = _run(empty, 20, 2048, 3, 0.05)
    assert bc.tolist() == [0, 0, 0] and np.isnan(bq).all()
    ws = torch.zeros((16,), dtype=torch.uint8, device=DEV)
    rc = B.sparrow_acceptance(inp["ids_p"], inp["logp_p"], inp["ids_q"], inp["logp_q"], inp["positions"], 20, 2048, 3, 0.05,
                              torch.zeros(1, device=DEV), torch.zeros(3, device=DEV), torch.zeros(3, dtype=torch.int32, device=DEV), ws, check=False)
    assert rc == -3
    rc = B.sparrow_acceptance(inp["ids_p"], inp["logp_p"], inp["ids_q"], inp["logp_q"], inp["positions"], 33, 2048, 3, 0.05,
                              torch.zeros(1, device=DEV), torch.zeros(3, device=DEV), torch.zeros(3, dtype=torch.int32, device=DEV), ws, check=False)
    assert rc == -1
