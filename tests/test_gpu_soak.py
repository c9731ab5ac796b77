"""Soak of the hand-rolled synchronisation (``-m gpu``; stands in for compute-sanitizer racecheck, which is closed on this
pool -- DESIGN.md 9).  decode_kernel coordinates nine warps through volatile shared-memory words, a descriptor ring with a
computed reuse distance, two parking areas handed out by generation number, and cross-CTA acquire/release counters that must
restore themselves to zero; select_kernel has its own arrival counters.  The parity tests call each shape once or a handful
of times: a slip with a 1e-4 hit rate would pass them and then trap a long rollout.  Here 8000 steps run back to back over
eight seeded batches (r in {1, 2, 5, 8}, pages of 16 and 64 tokens, units spanning many CTAs and hundreds of tiny units),
in the deterministic mode so that EVERY bit of every call is compared with the first call of its batch, and after every call
the self-restoring counters of both workspaces (sparrow.h: "the kernel restores the zeros it uses") are asserted zero.
The last call of each batch is checked against the oracle."""
import numpy as np
import pytest
import torch

from paper_2606_08446_b200 import binding as B
from paper_2606_08446_b200 import workloads as W

from parity_util import assert_same_result, check_sparse_step

pytestmark = pytest.mark.gpu
DEV = "cuda"

BATCHES = [   # (Hq, Hkv, page, lengths, budget tokens)
    (2, 2, 16, [1, 15, 16, 17, 33, 250, 256, 257, 1000, 2049, 4099], 200),
    (4, 2, 16, [33000, 9, 2500], 9000),
    (5, 1, 16, [20000, 17, 3, 9000, 12345], 6000),
    (8, 1, 16, [40000, 25000], 20000),
    (16, 8, 64, [6000, 300, 2500, 64, 65], 2048),
    (40, 8, 16, [5000, 4100, 77, 3001], 1024),
    (8, 2, 64, [30000, 1, 129], 8192),
    (8, 2, 16, "short700", 96),
]


def _batch(k):
    Hq, Hkv, page, lens, budget = BATCHES[k]
    if lens == "short700":
        lens = [int(x) for x in np.random.default_rng(100 + k).integers(1, 700, size=700)]
    sched = W._sched("fixed", 16, 64, fixed_tokens=budget)
    return W.make_workload(n_seq=len(lens), Hq=Hq, Hkv=Hkv, lengths=("list", lens), schedule=sched, seed=500 + k, device=DEV,
                           plant=True, poison_tail=True, page_size=page)


def _ctr_words(eng):
    """The counter regions at the head of the two workspaces: select -- one int32 per (sequence, kv-head) unit; decode -- the
    same plus the tail-piece counter and the CTAs-done counter."""
    units = eng.wl.n_seq * eng.wl.Hkv
    return eng.select_ws[: 4 * units].view(torch.int32), eng.sparse_ws[: 4 * (units + 2)].view(torch.int32), \
        eng.dense_ws[: 4 * (units + 2)].view(torch.int32)


@pytest.mark.parametrize("k", range(len(BATCHES)))
def test_soak_bitwise_repeat_and_workspaces_restored(k):
    from paper_2606_08446_b200.engine import SparrowEngine
    wl = _batch(k)
    eng = SparrowEngine(wl, deterministic=True, want_scores=True)
    eng.summarize_all()
    eng.step(); eng.dense_decode()
    torch.cuda.synchronize()
    ref = [t.clone() for t in (eng.sel_pages, eng.sel_count, eng.out, eng.lse, eng.out_dense, eng.lse_dense)]
    sel_c, dec_c, den_c = _ctr_words(eng)
    assert not sel_c.any() and not dec_c.any() and not den_c.any(), "counters not restored after the first call"
    n_steps = 1000
    # flags accumulated on the device; one sync every 50 steps keeps the launches back to back
    bad = torch.zeros((3,), dtype=torch.int64, device=DEV)
    for s in range(n_steps):
        eng.step()
        if s % 3 == 0:
            eng.dense_decode()
        bad[0] += (sel_c != 0).sum() + (dec_c != 0).sum() + (den_c != 0).sum()
        bad[1] += (eng.sel_pages != ref[0]).sum() + (eng.sel_count != ref[1]).sum()
        bad[2] += (eng.out != ref[2]).sum() + (eng.lse != ref[3]).sum() + (eng.out_dense != ref[4]).sum() + (eng.lse_dense != ref[5]).sum()
        if s % 50 == 49:
            b = bad.tolist()
            assert b[0] == 0, f"batch {k} step {s}: {b[0]} workspace counter words left non-zero"
            assert b[1] == 0, f"batch {k} step {s}: selection differs from the first call in {b[1]} entries"
            assert b[2] == 0, f"batch {k} step {s}: out / lse differ from the first call in {b[2]} entries"
    check_sparse_step(eng, wl, check_summ=False)


def test_soak_default_mode_keeps_its_workspaces_clean_too():
    """The run-time hand-out (default mode) over the same protocol: integer outputs bitwise, out to the arithmetic's error,
    counters zero after every call."""
    from paper_2606_08446_b200.engine import SparrowEngine
    for k in (1, 2, 7):
        wl = _batch(k)
        eng = SparrowEngine(wl)
        eng.summarize_all()
        eng.step()
        torch.cuda.synchronize()
        ref_sel, ref_cnt, ref_out, ref_lse = eng.sel_pages.clone(), eng.sel_count.clone(), eng.out.clone(), eng.lse.clone()
        sel_c, dec_c, _ = _ctr_words(eng)
        bad = torch.zeros((2,), dtype=torch.int64, device=DEV)
        for s in range(200):
            eng.step()
            bad[0] += (sel_c != 0).sum() + (dec_c != 0).sum()
            bad[1] += (eng.sel_pages != ref_sel).sum() + (eng.sel_count != ref_cnt).sum()
        assert bad.tolist() == [0, 0]
        assert_same_result(eng.out, ref_out, f"default-mode soak batch {k}", eng.lse, ref_lse)
        check_sparse_step(eng, wl, check_summ=False)
