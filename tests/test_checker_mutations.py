"""The parity checker itself (CPU, ``-m "not gpu"``): tests/parity_util.check_selection / check_outputs must REJECT a wrong
result, not only accept a right one.  Every GPU run on record has had differing_units = 0, so nothing so far showed that the
checker's validity rules bite.  Here the oracle's own cfg1 result stands in for the GPU output and is corrupted one way at a
time; each corruption must raise, and the one legitimate difference -- a swap inside the
R10 tie band -- must pass and be counted."""
import copy

import numpy as np
import pytest
import torch

import oracle
from paper_2606_08446_b200 import workloads as W

from parity_util import BAND_REL, check_outputs, check_selection


@pytest.fixture(scope="module")
def case():
    wl = W.make_config("cfg1", device="cpu")
    h = wl.host()
    sched = oracle.Schedule.from_spec(wl.schedule)
    res = oracle.sparse_step(h["q"], h["k_cache"], h["v_cache"], h["page_table"], h["seq_lens"], sched, wl.sm_scale, max_sel=16)
    return wl, h, sched, res


def _gpu_like(res):
    return res["sel"].copy(), res["sel_count"].astype(np.int32).copy()


def _candidates(res, h, i, g):
    """(selected top-k pages, unselected candidate pages) of unit (i, g), by the oracle."""
    L = int(h["seq_lens"][i]); n_pages = -(-L // 16)
    F = set(np.flatnonzero(res["forced"][i, :n_pages]).tolist())
    cnt = int(res["sel_count"][i])
    sel = set(res["sel"][i, g, :cnt].tolist())
    top = sorted(sel - F)
    rest = sorted(set(range(n_pages)) - sel)
    return top, rest, F


def test_the_oracles_own_result_passes(case):
    wl, h, sched, res = case
    sel, cnt = _gpu_like(res)
    st = check_selection(res, sel, cnt, h["seq_lens"], res["scores"].astype(np.float32))
    assert st == dict(units=4, differing_units=0, band_pages=0)
    out = torch.from_numpy(res["out"]).to(torch.bfloat16)
    check_outputs(out, torch.from_numpy(res["lse"]).float(), res["out"], res["lse"])


def test_a_candidate_outside_the_band_is_rejected(case):
    wl, h, sched, res = case
    sel, cnt = _gpu_like(res)
    top, rest, F = _candidates(res, h, 1, 0)
    worst = min(rest, key=lambda p: res["scores"][1, 0, p])              # far below the threshold
    row = sorted((set(sel[1, 0, :cnt[1]].tolist()) - {top[0]}) | {worst})
    sel[1, 0, :cnt[1]] = row
    with pytest.raises(AssertionError, match="outside the tie band"):
        check_selection(res, sel, cnt, h["seq_lens"])


def test_a_swap_inside_the_band_passes_and_is_counted(case):
    wl, h, sched, res = case
    res2 = copy.deepcopy(res)
    sel, cnt = _gpu_like(res2)
    top, rest, F = _candidates(res2, h, 0, 1)
    tau = res2["tau"][0, 1]
    kth = min(top, key=lambda p: res2["scores"][0, 1, p])                # the page at the threshold
    assert res2["scores"][0, 1, kth] == tau
    runner = max(rest, key=lambda p: res2["scores"][0, 1, p])
    res2["scores"][0, 1, runner] = tau * (1 - 0.5 * BAND_REL * np.sign(tau))   # a near tie the fp32 kernel may order either way
    sel[0, 1, :cnt[0]] = sorted((set(sel[0, 1, :cnt[0]].tolist()) - {kth}) | {runner})
    st = check_selection(res2, sel, cnt, h["seq_lens"])
    assert st["differing_units"] == 1 and st["band_pages"] == 2
    res2["scores"][0, 1, runner] = tau * (1 - 3.0 * BAND_REL * np.sign(tau))   # just outside: rejected
    with pytest.raises(AssertionError, match="outside the tie band"):
        check_selection(res2, sel, cnt, h["seq_lens"])


def test_a_dropped_forced_page_is_rejected(case):
    wl, h, sched, res = case
    sel, cnt = _gpu_like(res)
    top, rest, F = _candidates(res, h, 0, 0)
    sink = min(F)
    row = sorted((set(sel[0, 0, :cnt[0]].tolist()) - {sink}) | {rest[0]})
    sel[0, 0, :cnt[0]] = row
    with pytest.raises(AssertionError, match="forced pages missing"):
        check_selection(res, sel, cnt, h["seq_lens"])


def test_duplicates_disorder_range_and_count_are_rejected(case):
    wl, h, sched, res = case
    sel, cnt = _gpu_like(res)
    s2 = sel.copy(); s2[1, 1, 5] = s2[1, 1, 4]                           # duplicate
    with pytest.raises(AssertionError, match="strictly ascending"):
        check_selection(res, s2, cnt, h["seq_lens"])
    s2 = sel.copy(); s2[1, 1, [3, 4]] = s2[1, 1, [4, 3]]                 # two entries out of order
    with pytest.raises(AssertionError, match="strictly ascending"):
        check_selection(res, s2, cnt, h["seq_lens"])
    s2 = sel.copy(); s2[1, 1, cnt[1] - 1] = 94                           # one past the last page (L = 1500 -> pages 0..93)
    with pytest.raises(AssertionError, match="out of range"):
        check_selection(res, s2, cnt, h["seq_lens"])
    s2 = sel.copy(); s2[0, 0, 0] = -1
    with pytest.raises(AssertionError):
        check_selection(res, s2, cnt, h["seq_lens"])
    for d in (-1, 1):                                                    # count off by one
        c2 = cnt.copy(); c2[0] += d
        with pytest.raises(AssertionError, match="sel_count"):
            check_selection(res, sel, c2, h["seq_lens"])


def test_wrong_fp32_scores_are_rejected(case):
    wl, h, sched, res = case
    sel, cnt = _gpu_like(res)
    sc = res["scores"].astype(np.float32)
    top, rest, F = _candidates(res, h, 0, 0)
    sc[0, 0, rest[3]] *= 1.001
    with pytest.raises(AssertionError, match="fp32 scores off"):
        check_selection(res, sel, cnt, h["seq_lens"], sc)


def test_an_output_that_misses_one_page_is_rejected(case):
    """The failure the lse gate exists for: one selected page's tokens left out of (or counted twice in) a head's softmax."""
    wl, h, sched, res = case
    cnt = res["sel_count"].astype(np.int64)
    for mode in ("dropped", "doubled"):
        sel = res["sel"].copy()
        c2 = cnt.copy()
        if mode == "dropped":                                            # sequence 0 attends to 15 of its 16 pages
            sel[0, :, 7:15] = sel[0, :, 8:16]; c2[0] -= 1
            out, lse = oracle.attention_on_sets(h["q"], h["k_cache"], h["v_cache"], h["page_table"], h["seq_lens"], sel, c2, wl.sm_scale)
        else:                                                            # one page's tokens counted twice = its mass doubled
            out, lse = res["out"].copy(), res["lse"].copy()
            sel1 = sel.copy(); sel1[0, :, 0] = sel[0, :, 7]; c1 = cnt.copy(); c1[0] = 1
            o1, l1 = oracle.attention_on_sets(h["q"], h["k_cache"], h["v_cache"], h["page_table"], h["seq_lens"], sel1, c1, wl.sm_scale)
            m = np.maximum(lse[0], l1[0]); a, b = np.exp(lse[0] - m), np.exp(l1[0] - m)
            out[0] = (out[0] * a[:, None] + o1[0] * b[:, None]) / (a + b)[:, None]
            lse[0] = m + np.log(a + b)
        got = torch.from_numpy(out).to(torch.bfloat16)
        with pytest.raises(AssertionError):
            check_outputs(got, torch.from_numpy(lse).float(), res["out"], res["lse"])
        # the lse alone gives it away even if the output rows were right
        with pytest.raises(AssertionError, match="lse off"):
            check_outputs(torch.from_numpy(res["out"]).to(torch.bfloat16), torch.from_numpy(lse).float(), res["out"], res["lse"])
