"""sparrow_select_static: page selection for callers that cannot allocate device memory (``-m gpu``).

Some users of this library are handed device pointers for their inputs and outputs but have nothing to allocate a
workspace with: a custom op living inside a server whose memory pool already owns the whole GPU, a step in a decode loop
that must not stall on cudaMalloc, a foreign-language caller of the C ABI with no CUDA allocator binding.  For them the
library carries a fixed 4 MiB scratch array of its own and `sparrow_select_static` uses it in place of the `workspace`
argument of `sparrow_select`.

What is checked here: the static entry gives the same page lists, counts and scores as `sparrow_select` given a
caller-allocated workspace -- bit for bit, which is the bar every selection test in this suite uses (integer output, exact
tie-break, one deterministic fp32 score per page) -- on two calls in a row, and again after a call of a different shape has
left its own contents in the shared array; and a shape whose scratch would not fit is refused with its own status before
anything runs.  The file sorts last on purpose: `pytest -x` stops at the first failure, so a problem in this side entry
must not hide the parity tests.  It makes no assumption about what ran before it (first call on the device or not).
"""
import pytest
import torch

from paper_2606_08446_b200 import workloads as W

pytestmark = pytest.mark.gpu
DEV = "cuda"


def _reference(wl):
    """The existing path: summaries, then sparrow_select with a workspace the engine allocated with torch."""
    from paper_2606_08446_b200.engine import SparrowEngine
    eng = SparrowEngine(wl, want_scores=True)
    eng.summarize_all()
    eng.select()
    torch.cuda.synchronize()
    return eng


def _static_call(eng, wl):
    """One call of the no-allocation entry into fresh output buffers (poisoned so that untouched entries show)."""
    from paper_2606_08446_b200 import binding as B
    sel = torch.full_like(eng.sel_pages, -1)
    cnt = torch.full_like(eng.sel_count, -7)
    scores = torch.full_like(eng.scores, float("nan"))
    B.sparrow_select_static(wl.q, eng.summaries, wl.page_table, wl.seq_lens, eng.sched, sel, eng.max_sel, cnt, scores, eng.shape)
    assert B.sparrow_last_launch_count() == 1                 # the select kernel; the counter clear is a memset, not a kernel
    torch.cuda.synchronize()
    return sel, cnt, scores


def _assert_same(eng, got, what):
    sel, cnt, scores = got
    assert torch.equal(cnt, eng.sel_count), f"{what}: sel_count differs"
    assert torch.equal(sel, eng.sel_pages), f"{what}: sel_pages differs"
    # scores_dbg: candidate entries are written, the others keep their NaN -- same positions, same bits
    assert torch.equal(torch.isnan(scores), torch.isnan(eng.scores)), f"{what}: a different set of pages was scored"
    assert torch.equal(torch.nan_to_num(scores), torch.nan_to_num(eng.scores)), f"{what}: scores differ"


def test_static_scratch_select_matches_the_workspace_path_twice_in_a_row():
    # several selector slices per unit, ragged lengths, dense-in-sparse short sequences, planted pages
    wl_a = W.make_workload(n_seq=7, Hq=8, Hkv=4, lengths=("list", [3000, 9000, 513, 4100, 77, 2500, 16]),
                           schedule=W._sched("fixed", 64, 256, fixed_tokens=1024), seed=31, device=DEV, plant=True)
    # another shape (other head counts, other page-table width): leaves different counters / scores behind in the array
    wl_b = W.make_workload(n_seq=3, Hq=5, Hkv=1, lengths=("list", [20000, 40, 6000]),
                           schedule=W._sched("clamp_frac", 16, 64, f0_ppm=125000, floor_tokens=512), seed=32, device=DEV, plant=True)
    eng_a, eng_b = _reference(wl_a), _reference(wl_b)
    assert (eng_a.sel_count.cpu() < torch.tensor([-(-L // 16) for L in [3000, 9000, 513, 4100, 77, 2500, 16]])).any()   # really sparse
    _assert_same(eng_a, _static_call(eng_a, wl_a), "first call")
    _assert_same(eng_a, _static_call(eng_a, wl_a), "second call in a row")
    _assert_same(eng_b, _static_call(eng_b, wl_b), "other shape after it")
    _assert_same(eng_a, _static_call(eng_a, wl_a), "first shape again, after the other shape's leftovers")


def test_static_scratch_select_refuses_what_does_not_fit():
    from paper_2606_08446_b200 import binding as B
    wl = W.make_config("cfg1", device=DEV)
    eng = _reference(wl)
    limit = B.sparrow_select_static_bytes()
    assert limit == 4 << 20
    # the same pointers under a shape whose scratch would exceed the array: refused by size alone, nothing is launched
    big = B.make_shape(1024, 32, 8, 2048, wl.n_phys)
    assert B.sparrow_select_workspace_bytes(big) > limit
    rc = B.sparrow_select_static(wl.q, eng.summaries, wl.page_table, wl.seq_lens, eng.sched, eng.sel_pages, eng.max_sel,
                                 eng.sel_count, None, big, check=False)
    assert rc == -5 and "4 MiB" in B.sparrow_strerror(rc) and "sparrow_select" in B.sparrow_strerror(rc)
    with pytest.raises(B.SparrowError, match="built-in array"):
        B.sparrow_select_static(wl.q, eng.summaries, wl.page_table, wl.seq_lens, eng.sched, eng.sel_pages, eng.max_sel,
                                eng.sel_count, None, big)
    # a shape right under the limit is accepted by the size check (cfg1 itself is far below it)
    assert B.sparrow_select_workspace_bytes(eng.shape) <= limit
    _assert_same(eng, _static_call(eng, wl), "cfg1 after a refused call")
