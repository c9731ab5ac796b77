"""GPU parity of the rollout loop (``-m gpu``): sparrow_append (+ summarize on page fill) ->
sparrow_select -> sparrow_sparse_decode for T steps with the lengths on the device, eagerly (every step checked
against the oracle's rollout) and as ONE CUDA graph (page lists and counts identical to the eager run, outputs equal to within the arithmetic's error: the decode hands tiles out at run time)."""
import numpy as np
import pytest
import torch

import oracle
from paper_2606_08446_b200 import workloads as W

from parity_util import assert_same_result, check_outputs, check_selection, check_summaries

pytestmark = pytest.mark.gpu
DEV = "cuda"
T = 36
LENS = [250, 1023, 15, 2040, 4090]
SCHED = W._sched("table", 16, 48, table_pages=(6, 9, 14, 20, 20, 24, 24, 30, 40), bin_tokens=512)


def _setup():
    from paper_2606_08446_b200.engine import SparrowEngine
    wl = W.make_workload(n_seq=len(LENS), Hq=8, Hkv=2, lengths=("list", LENS), schedule=SCHED, seed=21, device=DEV,
                         reserve_tokens=T + 3, plant=True)
    eng = SparrowEngine(wl, want_scores=True)
    eng.summarize_all()
    eng.reserve(T)
    qs, ks, vs = W.make_rollout_inputs(wl, T, seed=5)
    return wl, eng, qs, ks, vs


def _bits(t):
    return t.contiguous().view(torch.int16).cpu().numpy().view(np.uint16)


def test_rollout_eager_every_step_matches_oracle_and_graph_replay_agrees():
    wl, eng, qs, ks, vs = _setup()
    h0 = wl.host()
    osched = oracle.Schedule.from_spec(SCHED)
    want, kc, vc = oracle.rollout(_bits(qs), _bits(ks), _bits(vs), h0["k_cache"], h0["v_cache"], h0["page_table"],
                                  h0["seq_lens"], osched, wl.sm_scale, max_sel=eng.max_sel)
    out = torch.zeros((T, wl.n_seq, wl.Hq, 128), dtype=torch.bfloat16, device=DEV)
    lse = torch.zeros((T, wl.n_seq, wl.Hq), dtype=torch.float32, device=DEV)
    differing = 0
    for t in range(T):
        eng.append(ks[t], vs[t])
        eng.select(qs[t])
        eng.sparse_decode(qs[t], out=out[t], lse=lse[t])
        torch.cuda.synchronize()
        st = want[t]
        assert eng.wl.seq_lens.cpu().tolist() == st["seq_lens"].tolist()
        sel, cnt = eng.sel_pages.cpu().numpy(), eng.sel_count.cpu().numpy()
        stats = check_selection(st, sel, cnt, st["seq_lens"], eng.scores.cpu().numpy())
        if stats["differing_units"]:
            differing += stats["differing_units"]
            ht = dict(k_cache=_bits(wl.k_cache), v_cache=_bits(wl.v_cache))
            sel_fix = np.where(np.arange(sel.shape[2])[None, None, :] < cnt[:, None, None], sel, 0)
            wo, wlse = oracle.attention_on_sets(_bits(qs[t]), ht["k_cache"], ht["v_cache"], h0["page_table"], st["seq_lens"],
                                                sel_fix, cnt.astype(np.int64), wl.sm_scale)
        else:
            wo, wlse = st["out"], st["lse"]
        check_outputs(out[t], lse[t], wo, wlse, f"rollout step {t}")
        if st["filled"]:     # summarize-on-fill: the landmarks of the pages that just filled, bit for bit
            check_summaries(eng.summaries, dict(k_cache=_bits(wl.k_cache)), np.array(st["filled"]), None)
    # the cache after T appends is the oracle's, bit for bit
    assert np.array_equal(_bits(wl.k_cache), kc) and np.array_equal(_bits(wl.v_cache), vc)
    assert sum(len(s["filled"]) for s in want) >= 8       # page fills did happen (15 -> 16, 1023 -> 1024, ...)

    # ---- the same T steps as one CUDA graph on a fresh copy of the batch ----
    wl2, eng2, qs2, ks2, vs2 = _setup()
    assert torch.equal(qs2, qs) and torch.equal(wl2.k_cache[wl2.page_table[0, 0].long()], torch.as_tensor(h0["k_cache"][h0["page_table"][0, 0]].view(np.int16)).view(torch.bfloat16).to(DEV))
    out2 = torch.zeros_like(out)
    lse2 = torch.zeros_like(lse)
    st = torch.cuda.Stream()
    with torch.cuda.stream(st):
        # warm-up outside the graph must not advance this batch: use a throw-away engine state
        g = torch.cuda.CUDAGraph()
        with torch.cuda.graph(g, stream=st):
            eng2.rollout(qs2, ks2, vs2, out2, lse2, stream=st)
        g.replay()
    st.synchronize()
    torch.cuda.synchronize()
    assert wl2.seq_lens.cpu().tolist() == [L + T for L in LENS]
    assert_same_result(out2, out, "rollout as one CUDA graph vs step by step", lse2, lse)
    assert torch.equal(wl2.k_cache, wl.k_cache) and torch.equal(eng2.summaries, eng.summaries)


def test_rollout_dense_branch_and_cumulative_cost():
    """Dense rollout (append -> dense decode) against the oracle, and the paper's cost claim on the token counts:
    the sparse loop attends O(B) tokens per step, the dense loop O(L)."""
    wl, eng, qs, ks, vs = _setup()
    h0 = wl.host()
    Td = 6
    want, _, _ = oracle.rollout(_bits(qs[:Td]), _bits(ks[:Td]), _bits(vs[:Td]), h0["k_cache"], h0["v_cache"], h0["page_table"],
                                h0["seq_lens"], None, wl.sm_scale)
    out = torch.zeros((Td, wl.n_seq, wl.Hq, 128), dtype=torch.bfloat16, device=DEV)
    lse = torch.zeros((Td, wl.n_seq, wl.Hq), dtype=torch.float32, device=DEV)
    eng.rollout(qs[:Td], ks[:Td], vs[:Td], out, lse, dense=True)
    torch.cuda.synchronize()
    for t in range(Td):
        check_outputs(out[t], lse[t], want[t]["out"], want[t]["lse"], f"dense rollout step {t}")
    from paper_2606_08446_b200 import binding as B
    sparse_tok = sum(16 * B.sparrow_sel_count(eng.sched, L + t + 1) for L in LENS for t in range(T))
    dense_tok = sum(L + t + 1 for L in LENS for t in range(T))
    assert sparse_tok < 0.35 * dense_tok
