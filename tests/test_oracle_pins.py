"""Pins for the fp64 CPU oracle (``-m "not gpu"``).

Each test checks ``oracle/`` against something other than itself: values worked by hand from the
definitions (tests/golden/), numpy brute force on tiny inputs written from the token-level
definitions, closed forms, invariants and special cases (SURVEY.md section 8(c) "what pins each part").
A plausible mistake in the oracle (dropped term, wrong sign/index, transposed operand, off-by-one in a
page boundary) fails at least one of them.
"""
import math
import os

import numpy as np
import pytest
import torch

import oracle
from paper_2606_08446_b200 import workloads as W

GOLD = os.path.join(os.path.dirname(__file__), "golden")
P, D = 16, 128


def f64(bits):
    """bf16 bit patterns -> float64 (exact)."""
    return (np.asarray(bits, dtype=np.uint16).astype(np.uint32) << 16).view(np.float32).astype(np.float64)


def bf16_bits(x):
    return torch.as_tensor(np.asarray(x, dtype=np.float32)).to(torch.bfloat16).view(torch.int16).numpy().view(np.uint16)


def tiny(n_seq=2, Hq=4, Hkv=2, lens=(70, 33), seed=0, sched=None, plant=False, **kw):
    sched = sched or W._sched("fixed", 16, 16, fixed_tokens=48)
    wl = W.make_workload(n_seq=n_seq, Hq=Hq, Hkv=Hkv, lengths=("list", list(lens)), schedule=sched,
                         plant=plant, seed=seed, **kw)
    return wl, wl.host()


# --------------------------------------------------------------- O2-O4 budget / forced ----
def _golden_rows():
    rows = []
    with open(os.path.join(GOLD, "budget_values.txt")) as f:
        for line in f:
            line = line.strip()
            if not line or line.startswith("#"):
                continue
            c, *v = line.split()
            rows.append((c, *map(int, v)))
    return rows


@pytest.mark.parametrize("row", _golden_rows(), ids=lambda r: f"{r[0]}-L{r[1]}")
def test_budget_and_forced_match_hand_worked_values(row):
    cfg, L, n_pages, B, K, n_forced, k, n_cand = row
    sched = oracle.Schedule.from_spec(W.CONFIGS[cfg]["schedule"])
    assert -(-L // P) == n_pages
    assert oracle.budget_tokens(sched, L) == B
    assert oracle.k_pages(sched, L) == K
    forced = oracle.forced_pages(L, sched.sink_tokens, sched.local_tokens)
    assert forced.sum() == n_forced
    assert max(0, K - n_forced) == k
    assert n_pages - n_forced == n_cand


def test_cfg1_forced_sets_by_hand():
    # L=1024 -> F = {0} U {60..63}; L=1500 -> F = {0} U {89..93}
    assert np.flatnonzero(oracle.forced_pages(1024, 16, 64)).tolist() == [0, 60, 61, 62, 63]
    assert np.flatnonzero(oracle.forced_pages(1500, 16, 64)).tolist() == [0, 89, 90, 91, 92, 93]


def test_table4_budget_identity():
    # PAPER.md:428-434 (Table 4, first row garbled "166-4" = "16-64"): all four configs are budget 1024
    for page, num in ((16, 64), (32, 32), (64, 16), (128, 8)):
        s = oracle.Schedule(kind="table", table_pages=[num], bin_tokens=2048)
        assert oracle.budget_tokens(s, 40000, page_size=page) == 1024
        assert oracle.k_pages(s, 40000, page_size=page) == num


def test_table_schedule_uses_2k_length_bins():
    # tokens grouped by position with 2K bin size; budget is a page count per bin
    s = oracle.Schedule(kind="table", table_pages=[10, 20, 30], bin_tokens=2048)
    assert oracle.k_pages(s, 2048) == 10 and oracle.k_pages(s, 2049) == 20
    assert oracle.k_pages(s, 4096) == 20 and oracle.k_pages(s, 4097) == 30
    assert oracle.k_pages(s, 99999) == 30            # beyond the table: last bin
    assert oracle.k_pages(s, 100) == 7               # B clamps to L: ceil(100/16) pages = dense


@pytest.mark.parametrize("seed", range(3))
def test_forced_pages_token_level_bruteforce(seed):
    rng = np.random.default_rng(seed)
    for _ in range(200):
        L = int(rng.integers(1, 700)); S = int(rng.integers(0, 80)); Wn = int(rng.integers(0, 200))
        n_pages = -(-L // P)
        want = np.zeros(n_pages, bool)
        for t in range(L):                       # token-level definition
            if t < S or t >= L - Wn:
                want[t // P] = True
        want[n_pages - 1] = True                 # the page of the current token is always kept
        got = oracle.forced_pages(L, S, Wn)
        assert np.array_equal(got, want), (L, S, Wn)


def test_budget_clamps_and_dense_boundary():
    # dense while the context fits the budget  =>  K_pages == n_pages iff B >= L (R13)
    for cfg in ("cfg2", "cfg3", "cfg5"):
        s = oracle.Schedule.from_spec(W.CONFIGS[cfg]["schedule"])
        for L in (1, 15, 16, 17, 1000, 2047, 2048, 2049, 5000):
            B = oracle.budget_tokens(s, L)
            assert B == min(L, max(B, s.floor_tokens)) and B <= L
            if L <= s.floor_tokens:
                assert oracle.k_pages(s, L) == -(-L // P)
    s = oracle.Schedule(kind="dense")
    assert oracle.k_pages(s, 1500) == 94


# ------------------------------------------------------------------------ O1 summaries ----
def test_summaries_bruteforce_and_bounds():
    wl, h = tiny(lens=(70, 33), seed=3)
    ids, nv = W.full_page_updates(wl)
    got = oracle.summarize(h["k_cache"], ids.numpy(), nv.numpy())
    K = f64(h["k_cache"])
    for u, (pid, v) in enumerate(zip(ids.tolist(), nv.tolist())):
        tile = K[pid][:, :v, :]                                   # [Hkv][valid][D]
        assert np.array_equal(got[u, :, 0], tile.min(axis=1))
        assert np.array_equal(got[u, :, 1], tile.max(axis=1))
        assert (got[u, :, 0][:, None, :] <= tile).all() and (tile <= got[u, :, 1][:, None, :]).all()
    # partial page really ignores the tail: n_valid=1 gives min == max == the first key
    one = oracle.summarize(h["k_cache"], ids.numpy()[:1], np.array([1], np.int32))
    assert np.array_equal(one[0, :, 0], K[ids[0]][:, 0, :]) and np.array_equal(one[0, :, 0], one[0, :, 1])


# --------------------------------------------------------------------------- O5 scores ----
def test_scores_numpy_bruteforce_and_closed_form_R5():
    wl, h = tiny(lens=(100, 64), seed=5)
    K, q = f64(h["k_cache"]), f64(h["q"])
    r = wl.Hq // wl.Hkv
    for i, L in enumerate(h["seq_lens"].tolist()):
        n_pages = -(-L // P)
        for g in range(wl.Hkv):
            s = oracle.scores_unit(h["q"][i], h["k_cache"], h["page_table"][i], L, g)
            for p in range(n_pages):
                valid = min(P, L - P * p)
                tile = K[h["page_table"][i, p], g, :valid]          # [valid][D]
                mn, mx = tile.min(0), tile.max(0)
                qs = q[i, g * r:(g + 1) * r]                        # [r][D]
                want = np.maximum(qs * mn, qs * mx).sum()
                assert s[p] == pytest.approx(want, rel=1e-13, abs=1e-12)
                # R5 closed form: sum_d (Q+ mx + Q- mn)
                qp, qm = np.clip(qs, 0, None).sum(0), np.clip(qs, None, 0).sum(0)
                assert s[p] == pytest.approx((qp * mx + qm * mn).sum(), rel=1e-12, abs=1e-11)
                # Quest upper bound: per head >= max_t q.k_t ; group sum >= max_t sum_h q_h.k_t
                dots = tile @ qs.T                                   # [valid][r]
                assert s[p] >= dots.sum(1).max() - 1e-9
                assert np.maximum(qs * mn, qs * mx).sum(1).min() >= -1e300   # finite
                for j in range(r):
                    assert np.maximum(qs[j] * mn, qs[j] * mx).sum() >= dots[:, j].max() - 1e-9


def test_score_of_page_with_identical_keys_is_exact_dot():
    wl, h = tiny(lens=(64,), n_seq=1, seed=7)
    kc = h["k_cache"].copy()
    ph = h["page_table"][0, 2]
    kc[ph, :, :, :] = kc[ph, :, :1, :]                               # all 16 keys of page 2 identical
    K, q = f64(kc), f64(h["q"])
    for g in range(wl.Hkv):
        s = oracle.scores_unit(h["q"][0], kc, h["page_table"][0], 64, g)
        want = sum(q[0, hq] @ K[ph, g, 0] for hq in range(g * 2, g * 2 + 2))
        assert s[2] == pytest.approx(want, rel=1e-13)


# ---------------------------------------------------------------------------- O6 top-k ----
def test_topk_bruteforce_lexsort_and_properties():
    rng = np.random.default_rng(11)
    for trial in range(200):
        n_pages = int(rng.integers(1, 60))
        s = rng.standard_normal(n_pages)
        if trial % 3 == 0:
            s = np.round(s)                                           # many exact ties
        forced = rng.random(n_pages) < 0.2
        forced[-1] = True
        K = int(rng.integers(0, n_pages + 3))
        sel, tau = oracle.select_unit(s, forced, K)
        if K >= n_pages:
            assert sel.tolist() == list(range(n_pages))
            continue
        cand = np.flatnonzero(~forced)
        k = min(max(0, K - forced.sum()), len(cand))
        order = cand[np.lexsort((cand, -s[cand]))]                    # score desc, then page asc
        want = np.sort(np.concatenate([np.flatnonzero(forced), order[:k]]))
        assert sel.tolist() == want.tolist()
        assert len(set(sel.tolist())) == len(sel) and (np.diff(sel) > 0).all()
        if k > 0:
            assert tau == s[order[k - 1]]
            assert (s[order[:k]] >= tau).all() and (s[order[k:]] <= tau).all()


def test_topk_zero_query_ties_go_to_lowest_pages():
    # q = 0 => every score is 0 => T = the k lowest-index candidates (pins the R10 tie-break)
    wl, h = tiny(lens=(40 * P,), n_seq=1, seed=1, sched=W._sched("fixed", 16, 32, fixed_tokens=10 * P))
    h["q"][:] = 0
    res = oracle.sparse_step(h["q"], h["k_cache"], h["v_cache"], h["page_table"], h["seq_lens"],
                             oracle.Schedule.from_spec(wl.schedule), wl.sm_scale)
    # forced = {0} U {38, 39}; k = 10 - 3 = 7 -> candidates 1..7
    assert res["sel"][0, 0, :10].tolist() == [0, 1, 2, 3, 4, 5, 6, 7, 38, 39]
    assert (res["scores"][0, :, :40] == 0).all()


def test_topk_recovers_planted_pages():
    # strong planting (R19 alternative, oracle self-test only): top-k must contain every planted candidate
    sched = W._sched("fixed", 16, 32, fixed_tokens=24 * P)
    wl = W.make_workload(n_seq=2, Hq=4, Hkv=2, lengths=("list", [100 * P, 77 * P + 5]), schedule=sched,
                         plant=True, plant_scale=40.0, plant_frac=0.08, seed=21)
    h = wl.host()
    res = oracle.sparse_step(h["q"], h["k_cache"], h["v_cache"], h["page_table"], h["seq_lens"],
                             oracle.Schedule.from_spec(sched), wl.sm_scale, do_attention=False)
    for i in range(2):
        cnt = int(res["sel_count"][i])
        assert cnt == 24
        for g in range(2):
            sel = set(res["sel"][i, g, :cnt].tolist())
            assert len(wl.planted[i][g]) >= 6
            assert set(wl.planted[i][g].tolist()) <= sel
            assert (res["sel"][i, g, cnt:] == -1).all()


# ------------------------------------------------------------------------ O8 attention ----
def _numpy_attention(h, i, g, pages, L, Hq, Hkv, scale):
    """Independent brute force: gather tokens, mask by position, plain softmax."""
    K, V, q = f64(h["k_cache"]), f64(h["v_cache"]), f64(h["q"])
    r = Hq // Hkv
    pt = h["page_table"][i]
    ks = np.concatenate([K[pt[p], g] for p in pages], 0)
    vs = np.concatenate([V[pt[p], g] for p in pages], 0)
    pos = np.concatenate([np.arange(p * P, p * P + P) for p in pages])
    keep = pos < L
    ks, vs = ks[keep], vs[keep]
    out, lse = [], []
    for hq in range(g * r, (g + 1) * r):
        z = (ks @ q[i, hq]) * scale
        w = np.exp(z - z.max())
        out.append((w / w.sum()) @ vs)
        lse.append(z.max() + np.log(w.sum()))
    return np.array(out), np.array(lse)


@pytest.mark.parametrize("lens", [(70, 33), (16, 17), (1, 48), (255, 256)])
def test_dense_attention_matches_numpy_softmax(lens):
    wl, h = tiny(lens=lens, seed=sum(lens), poison_tail=True)
    out, lse = oracle.dense_step(h["q"], h["k_cache"], h["v_cache"], h["page_table"], h["seq_lens"], wl.sm_scale)
    for i, L in enumerate(lens):
        for g in range(wl.Hkv):
            wo, wl_ = _numpy_attention(h, i, g, list(range(-(-L // P))), L, wl.Hq, wl.Hkv, wl.sm_scale)
            np.testing.assert_allclose(out[i, g * 2:(g + 1) * 2], wo, rtol=1e-11, atol=1e-13)
            np.testing.assert_allclose(lse[i, g * 2:(g + 1) * 2], wl_, rtol=1e-12)


def test_softmax_rows_sum_to_one_and_one_hot_v_gives_page_mass():
    wl, h = tiny(lens=(90,), n_seq=1, seed=9)
    pages = [0, 2, 5]
    out, lse, probs = oracle.attention_unit(h["q"][0], h["k_cache"], h["v_cache"], h["page_table"][0], 90,
                                            pages, 1, wl.sm_scale, want_probs=True)
    np.testing.assert_allclose(probs.sum(1), 1.0, rtol=1e-13)
    assert (probs[:, 2 * P + 10:] == 0).all()            # page 5 holds tokens 80..89 only
    # V = one-hot(page index) in channel c  =>  out[:, c] = attention mass on that page
    vc = np.zeros_like(h["v_cache"])
    one = bf16_bits([1.0])[0]
    for c, p in enumerate(pages):
        vc[h["page_table"][0, p], :, :, c] = one
    out2, _ = oracle.attention_unit(h["q"][0], h["k_cache"], vc, h["page_table"][0], 90, pages, 1, wl.sm_scale)
    for c in range(3):
        np.testing.assert_allclose(out2[:, c], probs[:, c * P:(c + 1) * P].sum(1), rtol=1e-12)


def test_zero_query_gives_mean_of_v_and_log_count():
    wl, h = tiny(lens=(75,), n_seq=1, seed=2)
    h["q"][:] = 0
    out, lse = oracle.dense_step(h["q"], h["k_cache"], h["v_cache"], h["page_table"], h["seq_lens"], wl.sm_scale)
    V = f64(h["v_cache"])
    for g in range(wl.Hkv):
        toks = np.concatenate([V[h["page_table"][0, p], g] for p in range(5)], 0)[:75]
        np.testing.assert_allclose(out[0, 2 * g], toks.mean(0), rtol=1e-12, atol=1e-14)
    np.testing.assert_allclose(lse, math.log(75), rtol=1e-13)


def test_chunked_partials_merged_by_lse_equal_single_pass():
    wl, h = tiny(lens=(16 * 9 + 1,), n_seq=1, seed=4)
    L = 16 * 9 + 1
    pages = [0, 1, 3, 4, 6, 9]
    args = (h["q"][0], h["k_cache"], h["v_cache"], h["page_table"][0], L)
    for g in range(wl.Hkv):
        full_out, full_lse = oracle.attention_unit(*args, pages, g, wl.sm_scale)
        # chunks incl. an empty one and one whose only page has a single valid token (page 9)
        chunks = [[0, 1], [], [3, 4, 6], [9]]
        parts = [oracle.attention_partial_unit(*args, c, g, wl.sm_scale) for c in chunks]
        assert parts[1][1].tolist() == [0.0, 0.0] and np.isneginf(parts[1][0]).all()
        for j in range(2):
            o, lse = oracle.lse_merge([p[0][j] for p in parts], [p[1][j] for p in parts],
                                      np.stack([p[2][j] for p in parts]))
            assert np.isfinite(o).all()
            np.testing.assert_allclose(o, full_out[j], rtol=1e-12, atol=1e-14)
            assert lse == pytest.approx(full_lse[j], rel=1e-13)
    # all-empty merge: no NaN
    o, lse = oracle.lse_merge([-np.inf], [0.0], np.zeros((1, D)))
    assert (o == 0).all() and lse == -np.inf


# --------------------------------------------------------------------------- end to end ----
def test_sparse_equals_dense_when_budget_covers_context():
    # PAPER.md:494-496 (L_dense): sparse == dense whenever L <= B   (BASELINE.json config 1, B >= L run)
    wl = W.make_config("cfg1_dense")
    h = wl.host()
    sched = oracle.Schedule.from_spec(wl.schedule)
    res = oracle.sparse_step(h["q"], h["k_cache"], h["v_cache"], h["page_table"], h["seq_lens"], sched, wl.sm_scale)
    out, lse = oracle.dense_step(h["q"], h["k_cache"], h["v_cache"], h["page_table"], h["seq_lens"], wl.sm_scale)
    assert res["sel_count"].tolist() == [64, 94]
    assert np.array_equal(res["out"], out) and np.array_equal(res["lse"], lse)
    assert np.isnan(res["tau"]).all()


def test_cfg1_sparse_structure_and_attention_on_sets():
    wl = W.make_config("cfg1")
    h = wl.host()
    sched = oracle.Schedule.from_spec(wl.schedule)
    res = oracle.sparse_step(h["q"], h["k_cache"], h["v_cache"], h["page_table"], h["seq_lens"], sched, wl.sm_scale)
    assert res["sel_count"].tolist() == [16, 16] and res["k_pages"].tolist() == [16, 16]
    for i, F in enumerate(([0, 60, 61, 62, 63], [0, 89, 90, 91, 92, 93])):
        for g in range(2):
            sel = res["sel"][i, g, :16]
            assert set(F) <= set(sel.tolist()) and (np.diff(sel) > 0).all()
            # every selected candidate scores >= tau >= every unselected candidate
            n_pages = -(-int(h["seq_lens"][i]) // P)
            s = res["scores"][i, g, :n_pages]
            cand_in = [p for p in sel if p not in F]
            cand_out = [p for p in range(n_pages) if p not in set(sel.tolist())]
            assert min(s[cand_in]) == res["tau"][i, g] and max(s[cand_out]) <= res["tau"][i, g]
            wo, wlse = _numpy_attention(h, i, g, sel.tolist(), int(h["seq_lens"][i]), 4, 2, wl.sm_scale)
            np.testing.assert_allclose(res["out"][i, 2 * g:2 * g + 2], wo, rtol=1e-11, atol=1e-13)
            np.testing.assert_allclose(res["lse"][i, 2 * g:2 * g + 2], wlse, rtol=1e-12)
    o2, l2 = oracle.attention_on_sets(h["q"], h["k_cache"], h["v_cache"], h["page_table"], h["seq_lens"],
                                      res["sel"], res["sel_count"], wl.sm_scale)
    assert np.array_equal(o2, res["out"]) and np.array_equal(l2, res["lse"])
    # sparse differs from dense (it is an approximation), but not wildly: same sign of lse gap
    _, lse_d = oracle.dense_step(h["q"], h["k_cache"], h["v_cache"], h["page_table"], h["seq_lens"], wl.sm_scale)
    assert (res["lse"] < lse_d).all()           # attending a strict subset of tokens lowers the log-sum-exp


def test_oracle_rejects_undersized_max_sel():
    wl = W.make_config("cfg1")
    h = wl.host()
    with pytest.raises(ValueError):
        oracle.sparse_step(h["q"], h["k_cache"], h["v_cache"], h["page_table"], h["seq_lens"],
                           oracle.Schedule.from_spec(wl.schedule), wl.sm_scale, max_sel=8)


# ------------------------------------------------------------------ 8(f)-1: rollout loop (append + grow) ----
def _rollout_case(T=40, reserve=64):
    lens = [250, 1023, 15, 2040]
    sched = W._sched("table", 16, 48, table_pages=(6, 9, 14), bin_tokens=512)      # budget steps up as L crosses 512, 1024
    wl = W.make_workload(n_seq=len(lens), Hq=4, Hkv=2, lengths=("list", lens), schedule=sched, seed=21, device="cpu",
                         reserve_tokens=reserve)
    qs, ks, vs = W.make_rollout_inputs(wl, T, seed=5)
    bits = lambda t: t.contiguous().view(torch.int16).numpy().view(np.uint16)
    return wl, wl.host(), bits(qs), bits(ks), bits(vs), sched


def test_rollout_append_places_tokens_by_position_bruteforce():
    """After T appends token j of sequence i sits at (page_table[i][j // 16], row j % 16): checked token by token
    against the step inputs with indexing written here, not the oracle's (the cache a decode grows)."""
    T = 40
    wl, h, qs, ks, vs, sched = _rollout_case(T)
    steps, kc, vc = oracle.rollout(qs, ks, vs, h["k_cache"], h["v_cache"], h["page_table"], h["seq_lens"],
                                   oracle.Schedule.from_spec(sched), wl.sm_scale)
    for i, L0 in enumerate(h["seq_lens"].tolist()):
        assert steps[-1]["seq_lens"][i] == L0 + T
        for t in range(T):
            j = L0 + t
            page = h["page_table"][i, j // P]
            assert np.array_equal(kc[page, :, j % P, :], ks[t, i]) and np.array_equal(vc[page, :, j % P, :], vs[t, i])
        for j in range(0, L0, 97):       # old tokens untouched
            page = h["page_table"][i, j // P]
            assert np.array_equal(kc[page, :, j % P, :], h["k_cache"][page, :, j % P, :])
    # pages reported as filled are exactly those whose last row was written at that step
    for t, st in enumerate(steps):
        want = sorted(int(h["page_table"][i, (L0 + t) // P]) for i, L0 in enumerate(h["seq_lens"].tolist()) if (L0 + t + 1) % P == 0)
        assert sorted(st["filled"]) == want


def test_rollout_step_equals_one_shot_on_the_grown_cache_and_budget_follows_length():
    """Step t of the loop is O1..O8 on the cache as it stands after t + 1 appends (checked against a cache rebuilt
    here from scratch), and the attended-token count per step is the closed form of the TABLE schedule in 512-token
    bins -- the budget steps up when L crosses a bin edge and attention cost is O(B), not O(L)
    (PAPER.md:140, :498)."""
    T = 24
    wl, h, qs, ks, vs, sched = _rollout_case(T)
    osched = oracle.Schedule.from_spec(sched)
    steps, _, _ = oracle.rollout(qs, ks, vs, h["k_cache"], h["v_cache"], h["page_table"], h["seq_lens"], osched, wl.sm_scale)
    table, bins = sched["table_pages"], sched["bin_tokens"]
    for t in (0, 7, T - 1):
        kc, vc = h["k_cache"].copy(), h["v_cache"].copy()
        lens = h["seq_lens"].copy()
        for u in range(t + 1):
            for i in range(wl.n_seq):
                j = int(lens[i]); page = h["page_table"][i, j // P]
                kc[page, :, j % P] = ks[u, i]; vc[page, :, j % P] = vs[u, i]
                lens[i] += 1
        one = oracle.sparse_step(qs[t], kc, vc, h["page_table"], lens, osched, wl.sm_scale)
        assert np.array_equal(one["sel"], steps[t]["sel"]) and np.allclose(one["out"], steps[t]["out"], rtol=0, atol=1e-12)
        for i in range(wl.n_seq):
            L = int(lens[i]); n_pages = -(-L // P)
            budget_pages = table[min((L - 1) // bins, len(table) - 1)]
            n_forced = len(set(range(min(1, n_pages))) | set(range(max(L - 48, 0) // P, n_pages)))
            want = n_pages if budget_pages >= n_pages else max(budget_pages, n_forced)
            assert steps[t]["sel_count"][i] == want, (t, i, L)
    # sequence 1 (L0 = 1023) crosses the 1024 bin edge after its second append: 9 -> 14 pages
    assert steps[0]["sel_count"][1] == 9 and steps[1]["sel_count"][1] == 14


def test_rollout_dense_branch_is_dense_attention_on_the_grown_cache():
    T = 5
    wl, h, qs, ks, vs, sched = _rollout_case(T)
    steps, kc, vc = oracle.rollout(qs, ks, vs, h["k_cache"], h["v_cache"], h["page_table"], h["seq_lens"], None, wl.sm_scale)
    i, L = 2, int(h["seq_lens"][2]) + T                      # the 15-token sequence: numpy softmax over its 20 tokens
    keys = np.stack([f64(kc[h["page_table"][i, j // P], :, j % P, :]) for j in range(L)])      # [L][Hkv][D]
    vals = np.stack([f64(vc[h["page_table"][i, j // P], :, j % P, :]) for j in range(L)])
    q = f64(qs[T - 1, i])                                     # [Hq][D]
    for hq in range(wl.Hq):
        g = hq // (wl.Hq // wl.Hkv)
        z = keys[:, g, :] @ q[hq] * wl.sm_scale
        p = np.exp(z - z.max()); p /= p.sum()
        assert np.allclose(p @ vals[:, g, :], steps[-1]["out"][i, hq], rtol=0, atol=1e-12)


# ------------------------------------------------------------------ 8(f)-4: the paper's cost model ----
def test_cost_model_against_per_step_sums_and_limits():
    """App. F's closed forms against the per-decode-step sums they stand for, written out here:
    step t attends min(L_in + t, K) tokens (K and V: 2 elements x D each), and scores (L_in + t) / pagesize landmarks
    when L_in + t > K.  The closed forms are the continuous versions: they differ from the sums by the O(L) terms."""
    P_, B_, N_, D_, r_, I_, ps = 1.7e9, 4.0, 8.0, 128.0, 2.0, 300.0, 16.0
    for L_in, L_out, K in [(1000.0, 30000.0, 4096.0), (0.0, 5000.0, 1024.0), (6000.0, 2000.0, 4096.0), (100.0, 500.0, 4096.0)]:
        c = oracle.cost_model(P_, B_, N_, L_in, L_out, D_, r_, I_, K, ps, c=2.0)
        steps = np.arange(1, int(L_out) + 1, dtype=np.float64)
        ctx = L_in + steps
        attn_sum = 2 * np.minimum(ctx, K).sum()                     # K and V tokens over the rollout
        dense_sum = 2 * ctx.sum()
        visits = (ctx[ctx > K] / ps).sum()
        assert abs(c["attn_elems_dense"] - dense_sum) <= 2 * L_out
        assert abs(c["attn_elems_sparse"] - attn_sum) <= 2 * L_out
        assert abs(c["landmark_visits"] - visits) <= (L_in + L_out) / ps
        # memory and compute terms are those element counts times D (and r, B, N) plus the parameter terms
        assert math.isclose(c["sparse_mem"], 2 * P_ * L_out + B_ * N_ * D_ * c["attn_elems_sparse"], rel_tol=1e-15)
        assert math.isclose(c["dense_comp"], 2 * P_ * B_ * N_ * L_out + r_ * B_ * N_ * D_ * c["attn_elems_dense"], rel_tol=1e-15)
        assert math.isclose(c["scoring_mem"], 2.0 * B_ * N_ * D_ * c["landmark_visits"], rel_tol=1e-15)
        assert math.isclose(c["sparse_total"], c["sparse_comp"] + c["scoring_comp"] + I_ * (c["sparse_mem"] + c["scoring_mem"]), rel_tol=1e-15)
    # Eq. 3's two clean scoring terms as PRINTED at PAPER.md:142 (L_in = 0, one landmark vector per page, B = 1):
    #   compute r N D L_out^2 / (2 pagesize),  memory (before I) N D L_out^2 / (2 pagesize).
    # The calculator leaves out the K dense steps at the start (App. F's L_dense), i.e. a factor 1 - (K / L_out)^2.
    for L_out, K in [(32768.0, 16.0), (20000.0, 2048.0)]:
        c = oracle.cost_model(0.0, 1.0, N_, 0.0, L_out, D_, r_, I_, K, ps, c=1.0)
        under_budget = 1.0 - (K / L_out) ** 2
        assert math.isclose(c["scoring_comp"], r_ * N_ * D_ * L_out ** 2 / (2 * ps) * under_budget, rel_tol=1e-12)
        assert math.isclose(c["scoring_mem"], N_ * D_ * L_out ** 2 / (2 * ps) * under_budget, rel_tol=1e-12)
    c = oracle.cost_model(0.0, 1.0, N_, 0.0, 32768.0, D_, r_, I_, 16.0, ps, c=1.0)
    assert math.isclose(c["scoring_comp"], r_ * N_ * D_ * 32768.0 ** 2 / (2 * ps), rel_tol=1e-6)      # K << L_out: the printed term
    # the same r : 1 compute-to-memory ratio as the attention terms (Eq. 3's 2 r N D B L_out vs 2 I N D B L_out), any c
    c2 = oracle.cost_model(P_, B_, N_, 500.0, 9000.0, D_, r_, I_, 1024.0, ps, c=2.0)
    assert math.isclose(c2["scoring_comp"], r_ * c2["scoring_mem"], rel_tol=1e-15)
    assert math.isclose(c2["sparse_comp"] - 2 * P_ * B_ * N_ * 9000.0, r_ * (c2["sparse_mem"] - 2 * P_ * 9000.0), rel_tol=1e-12)
    # budget covers the whole context: sparse == dense, nothing is scored
    c = oracle.cost_model(P_, B_, N_, 100.0, 500.0, D_, r_, I_, 4096.0, ps)
    assert c["attn_elems_sparse"] == c["attn_elems_dense"] and c["landmark_visits"] == 0 and c["sparse_total"] == c["dense_total"]
    # O(K L_out) instead of O(L_out^2): doubling L_out doubles the budgeted part, quadruples the dense one
    a = oracle.cost_model(0, 1, 1, 0.0, 20000.0, D_, r_, I_, 1000.0, ps)
    b = oracle.cost_model(0, 1, 1, 0.0, 40000.0, D_, r_, I_, 1000.0, ps)
    assert math.isclose(b["attn_elems_dense"] / a["attn_elems_dense"], 4.0)
    assert 2.0 < b["attn_elems_sparse"] / a["attn_elems_sparse"] < 2.06
    # Table 4's configurations all have budget 1024: equal attention cost, scoring cost ~ 1/pagesize
    base = [oracle.cost_model(0, 1, 1, 16384.0, 1.0, D_, r_, I_, ps_ * n_, ps_) for ps_, n_ in ((16., 64.), (32., 32.), (64., 16.), (128., 8.))]
    assert len({x["attn_elems_sparse"] for x in base}) == 1
    assert math.isclose(base[0]["landmark_visits"] / base[3]["landmark_visits"], 8.0)


# ------------------------------------------------------------------ 8(f)-2: page sizes 32 / 64 / 128 (Table 4) ----
@pytest.mark.parametrize("page", [32, 64, 128])
def test_page_size_variants_whole_step_against_numpy_token_level(page):
    """The oracle at page sizes other than 16 (16-64, 32-32, 64-16, 128-8 all mean budget 1024)
    against a numpy restatement of the whole step written here at TOKEN level: summaries as min / max over each page's
    valid tokens, score = sum over the group's heads and channels of max(q*mn, q*mx), forced = pages touching the
    sink tokens, the last `W` tokens or the last token, top-k by (score desc, page asc), softmax over the valid tokens
    of the kept pages."""
    lens = [700, 129, 2000 + page // 2]
    S, Wn, budget = 40, 200, 8 * page                      # budget in tokens: 8 pages whatever the page size
    sched = W._sched("fixed", S, Wn, fixed_tokens=budget)
    wl = W.make_workload(n_seq=3, Hq=4, Hkv=2, lengths=("list", lens), schedule=sched, seed=31 + page, device="cpu",
                         page_size=page, plant=True)
    h = wl.host()
    assert h["k_cache"].shape[2] == page
    res = oracle.sparse_step(h["q"], h["k_cache"], h["v_cache"], h["page_table"], h["seq_lens"], oracle.Schedule.from_spec(sched),
                             wl.sm_scale)
    Kf, Vf, Qf = f64(h["k_cache"]), f64(h["v_cache"]), f64(h["q"])
    r = wl.Hq // wl.Hkv
    for i, L in enumerate(lens):
        n_pages = -(-L // page)
        tok_page = np.arange(L) // page
        forced = set(tok_page[:min(S, L)].tolist()) | set(tok_page[max(L - Wn, 0):].tolist()) | {int(tok_page[-1])}
        K_pages = min(-(-min(budget, L) // page), n_pages)
        want_cnt = n_pages if K_pages >= n_pages else max(K_pages, len(forced))
        assert res["sel_count"][i] == want_cnt
        for g in range(wl.Hkv):
            keys = np.stack([Kf[h["page_table"][i, t // page], g, t % page] for t in range(L)])      # [L][D]
            vals = np.stack([Vf[h["page_table"][i, t // page], g, t % page] for t in range(L)])
            qg = Qf[i, g * r:(g + 1) * r]                                                              # [r][D]
            score = np.full(n_pages, -np.inf)
            for p in range(n_pages):
                kp = keys[p * page:min((p + 1) * page, L)]
                mn, mx = kp.min(0), kp.max(0)
                score[p] = np.maximum(qg * mn, qg * mx).sum()
            if K_pages >= n_pages:
                keep = list(range(n_pages))
            else:
                cand = [p for p in range(n_pages) if p not in forced]
                k = max(0, K_pages - len(forced))
                order = sorted(cand, key=lambda p: (-score[p], p))[:k]
                keep = sorted(forced | set(order))
                assert np.allclose(res["scores"][i, g, cand], score[cand], rtol=1e-12, atol=1e-9)
            assert res["sel"][i, g, :want_cnt].tolist() == keep
            tok = np.concatenate([np.arange(p * page, min((p + 1) * page, L)) for p in keep])
            for hh in range(r):
                z = keys[tok] @ qg[hh] * wl.sm_scale
                pr = np.exp(z - z.max()); pr /= pr.sum()
                assert np.allclose(pr @ vals[tok], res["out"][i, g * r + hh], rtol=0, atol=1e-12)
                assert abs(z.max() + math.log(np.exp(z - z.max()).sum()) - res["lse"][i, g * r + hh]) < 1e-12


# ------------------------------------------------------------------ 8(f)-3: acceptance rate (Eq. 1) and its tail ----
def test_acceptance_rate_eq1_identity_and_special_cases():
    """PAPER.md:76-79 Eq. 1: with the lists covering the whole vocabulary, alpha = sum_x min(p, q) must equal the
    expectation form E_{x~Q}[min(p/q, 1)] and 1 - total-variation distance, both computed here from the definitions;
    identical policies give 1, disjoint supports give 0; list order does not matter."""
    rng = np.random.default_rng(3)
    V, n = 50, 40
    lp = rng.normal(size=(n, V)); lq = lp + 0.7 * rng.normal(size=(n, V))
    lp -= np.log(np.exp(lp).sum(1, keepdims=True)); lq -= np.log(np.exp(lq).sum(1, keepdims=True))
    ids = np.tile(np.arange(V), (n, 1))
    perm = np.stack([rng.permutation(V) for _ in range(n)])
    a = oracle.acceptance_rate(ids, lp, np.take_along_axis(ids, perm, 1), np.take_along_axis(lq, perm, 1))
    p, q = np.exp(lp), np.exp(lq)
    assert np.allclose(a, (q * np.minimum(p / q, 1.0)).sum(1), rtol=0, atol=1e-14)           # expectation under Q
    assert np.allclose(a, 1.0 - 0.5 * np.abs(p - q).sum(1), rtol=0, atol=1e-14)             # 1 - TV distance
    assert np.allclose(oracle.acceptance_rate(ids, lp, ids, lp), 1.0, atol=1e-14)
    assert np.all(oracle.acceptance_rate(ids[:, :20], lp[:, :20], ids[:, 25:45], lq[:, 25:45]) == 0.0)
    # truncated lists: only shared tokens count (R23): here exactly tokens 10..19
    got = oracle.acceptance_rate(ids[:, :20], lp[:, :20], ids[:, 10:30], lq[:, 10:30])
    assert np.allclose(got, np.minimum(p[:, 10:20], q[:, 10:20]).sum(1), atol=1e-15)


def test_binned_quantile_is_the_nearest_rank_quantile():
    """The 5-percentile per 2K-position bin against numpy's own inverted-CDF quantile, and the
    bin edges / empty bins by hand."""
    rng = np.random.default_rng(4)
    pos = rng.integers(0, 9000, size=5000)
    alpha = rng.beta(8, 1, size=5000)
    counts, qv = oracle.binned_quantile(alpha, pos, 2048, 6, 0.05)
    for b in range(6):
        sel = alpha[np.minimum(pos // 2048, 5) == b]
        assert counts[b] == len(sel)
        if len(sel):
            assert qv[b] == np.quantile(sel, 0.05, method="inverted_cdf")
        else:
            assert np.isnan(qv[b])
    assert counts[5] == 0 and counts[4] == (pos >= 8192).sum()
    c, v = oracle.binned_quantile([0.5, 0.1, 0.9, 0.3], [0, 2047, 2048, 5000], 2048, 2, 0.5)
    assert c.tolist() == [2, 2] and v.tolist() == [0.1, 0.3]                                  # rank ceil(0.5 * 2) = 1


# ------------------------------------------------------------------ 8(f)-2: the mean-key landmark ----
def _bf16_neighbours(x: float):
    """The two bf16 values that bracket x (found by truncating the fp32 pattern; independent of the oracle's rounding)."""
    f = np.array([x], dtype=np.float32)
    lo_bits = f.view(np.uint32) & np.uint32(0xFFFF0000)
    cands = []
    for d in (-1, 0, 1, 2):
        b = (lo_bits.astype(np.int64) + d * 0x10000).astype(np.uint32)
        cands.append((float(b.view(np.float32)[0]), int(b[0] >> 16)))
    return cands


def test_mean_landmark_is_the_exact_mean_rounded_once():
    """summarize_mean = the arithmetic mean of the page's valid keys rounded ONCE to bf16 (reading R24; PAPER.md:142's
    one vector per page).  Pinned with exact rational arithmetic (fractions.Fraction, no floating point at all): the
    returned code is the bf16 value nearest to the exact mean -- nearer than every neighbouring code, ties to the even
    code -- and on the special cases: one valid token -> that key; identical keys -> that key; mean_landmark_band's
    exact mean == the rational mean to fp64 precision."""
    from fractions import Fraction
    wl = W.make_workload(n_seq=2, Hq=4, Hkv=2, lengths=("list", [100, 37]), schedule=W._sched("dense", 0, 0), seed=77, device="cpu")
    h = wl.host()
    ids = np.array([0, 3, 5, 2], np.int32)
    nv = np.array([16, 1, 9, 16], np.int32)
    got = oracle.summarize_mean(h["k_cache"], ids, nv)
    exact64, err = oracle.mean_landmark_band(h["k_cache"], ids, nv)
    kf = f64(h["k_cache"])
    for u, (pg, v) in enumerate(zip(ids, nv)):
        for g in range(2):
            for d in range(0, 128, 5):
                mean = sum(Fraction(float(kf[pg, g, t, d])) for t in range(v)) / int(v)       # exact
                code = int(got[u, g, d])
                val = Fraction(float(f64(np.array([code], np.uint16))[0]))
                dist = abs(val - mean)
                for nb_val, nb_code in _bf16_neighbours(float(mean)):
                    if nb_code == code:
                        continue
                    nd = abs(Fraction(nb_val) - mean)
                    assert dist < nd or (dist == nd and code % 2 == 0), (u, g, d, code, nb_code)
                assert abs(Fraction(float(exact64[u, g, d])) - mean) <= Fraction(2.0 ** -50) * abs(mean) + Fraction(2.0 ** -1000)
                assert err[u, g, d] >= 0 and err[u, g, d] <= (v + 1) * 2.0 ** -24 * float(np.abs(kf[pg, g, :v, d]).max()) * 1.0000001
    assert np.array_equal(got[1], h["k_cache"][3][:, 0, :])                              # one valid token
    kc = h["k_cache"].copy(); kc[7, :, :, :] = kc[7, :, :1, :]
    assert np.array_equal(oracle.summarize_mean(kc, np.array([7], np.int32))[0], kc[7][:, 0, :])
    # an fp32 running sum in token order (what a kernel does) lands on the same code or one step away, and only near a boundary
    for u, (pg, v) in enumerate(zip(ids, nv)):
        k32 = (wl.k_cache[int(pg)].float()[:, :v, :].cumsum(1)[:, -1, :] / float(v)).to(torch.bfloat16).view(torch.int16).numpy().view(np.uint16)
        diff = k32.astype(np.int64) - got[u].astype(np.int64)
        assert (np.abs(diff) <= 1).all()
        for g, d in zip(*np.nonzero(diff)):
            mid = 0.5 * (f64(np.array([k32[g, d]], np.uint16))[0] + f64(np.array([got[u, g, d]], np.uint16))[0])
            assert abs(exact64[u, g, d] - mid) <= err[u, g, d]


def test_mean_landmark_step_against_numpy_token_level():
    """The whole step with the mean-key landmark (PAPER.md:142's one vector per page) against a restatement written
    here: fp64 mean per page rounded to the nearer of its two bracketing bf16 values, score = (sum of the group's queries) . mean, top-k by (score desc, page asc) among the
    non-forced pages, softmax over the kept pages' valid tokens; plus planted pages recovered and B >= L == dense."""
    lens = [700, 129, 2050]
    S, Wn, budget = 40, 200, 256
    sched = W._sched("fixed", S, Wn, fixed_tokens=budget)
    wl = W.make_workload(n_seq=3, Hq=4, Hkv=2, lengths=("list", lens), schedule=sched, seed=91, device="cpu", plant=True, plant_scale=6.0)
    h = wl.host()
    res = oracle.sparse_step_mean(h["q"], h["k_cache"], h["v_cache"], h["page_table"], h["seq_lens"], oracle.Schedule.from_spec(sched), wl.sm_scale)
    Kf, Vf, Qf = f64(h["k_cache"]), f64(h["v_cache"]), f64(h["q"])
    r = wl.Hq // wl.Hkv
    for i, L in enumerate(lens):
        n_pages = -(-L // P)
        forced = set(range(min(3, n_pages))) | set(range(max(L - Wn, 0) // P, n_pages))  # 40 sink tokens = 3 pages
        dense_seq = budget // P >= n_pages
        assert res["sel_count"][i] == (n_pages if dense_seq else max(budget // P, len(forced)))
        for g in range(wl.Hkv):
            qsum = Qf[i, g * r:(g + 1) * r].sum(0)
            score = np.zeros(n_pages)
            for p in range(n_pages):
                v = min(P, L - p * P)
                mean = Kf[int(h["page_table"][i, p]), g, :v].mean(0)
                m = np.array([min(_bf16_neighbours(float(x)), key=lambda c: (abs(c[0] - x), c[1] % 2))[0] for x in mean])
                score[p] = m @ qsum
            cand = [p for p in range(n_pages) if p not in forced]
            keep = list(range(n_pages)) if dense_seq else sorted(forced | set(sorted(cand, key=lambda p: (-score[p], p))[:max(0, budget // P - len(forced))]))
            assert res["sel"][i, g, :len(keep)].tolist() == keep
            planted = [p for p in wl.planted[i][g].tolist() if p not in forced]
            if not dense_seq:
                assert len(set(planted) & set(keep)) >= min(len(planted), max(0, budget // P - len(forced))) - 1
            tok = np.concatenate([np.arange(p * P, min((p + 1) * P, L)) for p in keep])
            keys = np.stack([Kf[h["page_table"][i, t // P], g, t % P] for t in tok])
            vals = np.stack([Vf[h["page_table"][i, t // P], g, t % P] for t in tok])
            for hh in range(r):
                z = keys @ Qf[i, g * r + hh] * wl.sm_scale
                pr = np.exp(z - z.max()); pr /= pr.sum()
                assert np.allclose(pr @ vals, res["out"][i, g * r + hh], rtol=0, atol=1e-12)
    big = oracle.sparse_step_mean(h["q"], h["k_cache"], h["v_cache"], h["page_table"], h["seq_lens"],
                                  oracle.Schedule.from_spec(W._sched("fixed", S, Wn, fixed_tokens=4096)), wl.sm_scale)
    dense_out, dense_lse = oracle.dense_step(h["q"], h["k_cache"], h["v_cache"], h["page_table"], h["seq_lens"], wl.sm_scale)
    assert np.allclose(big["out"], dense_out, rtol=0, atol=1e-12) and np.allclose(big["lse"], dense_lse, rtol=0, atol=1e-12)
