"""GPU parity tests (``-m gpu``): the CUDA library, called through the C ABI binding, against the fp64 oracle,
element by element on the same seeded inputs.  Sizes span several tiles / chunks and ragged tails; the
full-size BASELINE.json configs (2, 3, 4, 5) are checked in the launch configuration bench.py times: selection on
every sequence, outputs on every sequence (cfg4: every sequence of one K/V pool)."""
import numpy as np
import pytest
import torch

import oracle
from paper_2606_08446_b200 import workloads as W

from parity_util import assert_same_result, check_dense, check_sparse_step, check_summaries, check_outputs, sub_host

pytestmark = pytest.mark.gpu
DEV = "cuda"


def _engine(wl, **kw):
    from paper_2606_08446_b200.engine import SparrowEngine
    eng = SparrowEngine(wl, **kw)
    eng.summarize_all()
    return eng


def _run_sparse(wl, **kw):
    eng = _engine(wl, **kw)
    eng.select()
    eng.sparse_decode()
    torch.cuda.synchronize()
    return eng


def test_library_loaded_is_in_tree():
    from paper_2606_08446_b200 import binding as B
    assert B.LIB_PATH.endswith("paper_2606_08446_b200/libsparrow_b200.so") and B.sparrow_version() >= 100


def test_cfg1_sparse_matches_oracle():
    wl = W.make_config("cfg1", device=DEV)
    eng = _run_sparse(wl, want_scores=True)
    st = check_sparse_step(eng, wl)
    assert eng.sel_count.tolist() == [16, 16]
    assert st["units"] == 4


def test_cfg1_budget_covers_context_equals_dense():
    wl = W.make_config("cfg1_dense", device=DEV)
    eng = _run_sparse(wl)
    st = check_sparse_step(eng, wl)
    assert eng.sel_count.tolist() == [64, 94] and st["differing_units"] == 0
    eng.dense_decode()
    torch.cuda.synchronize()
    check_dense(eng, wl)
    # sparse entry with B >= L vs dense entry: same tolerances (bitwise equality not required)
    assert (eng.out.float() - eng.out_dense.float()).abs().max().item() <= 2e-2
    assert (eng.lse - eng.lse_dense).abs().max().item() <= 1e-3


@pytest.mark.parametrize("Hq,Hkv", [(2, 2), (4, 2), (8, 2), (5, 1), (16, 2), (40, 8)])
def test_ragged_lengths_all_group_sizes(Hq, Hkv):
    lens = [1, 15, 16, 17, 33, 250, 256, 257, 1000, 2049, 4099]
    sched = W._sched("fixed", 16, 64, fixed_tokens=200)
    wl = W.make_workload(n_seq=len(lens), Hq=Hq, Hkv=Hkv, lengths=("list", lens), schedule=sched, seed=Hq * 100 + Hkv,
                         device=DEV, poison_tail=True, plant=True)
    eng = _run_sparse(wl, want_scores=True)
    check_sparse_step(eng, wl)
    eng.dense_decode()
    torch.cuda.synchronize()
    check_dense(eng, wl)


@pytest.mark.parametrize("Hq,Hkv,lens,budget", [(8, 2, [33000], 9000), (5, 1, [20000, 17], 6000), (16, 8, [40000, 3, 25000], 20000)])
def test_units_that_span_many_ctas(Hq, Hkv, lens, budget):
    """Few, very long units: the decode stream of ONE (sequence, kv-head) unit is cut over tens of CTAs (up to all 148), so
    the cross-piece merge (a7) folds tens of partials -- its multi-round loop, the last-arriver's register path and the
    workspace slots unit + piece id -- where the full-size configs only ever see two or three pieces per unit."""
    sched = W._sched("fixed", 64, 512, fixed_tokens=budget)
    wl = W.make_workload(n_seq=len(lens), Hq=Hq, Hkv=Hkv, lengths=("list", lens), schedule=sched, seed=Hq * 7 + Hkv, device=DEV,
                         poison_tail=True, plant=True)
    eng = _run_sparse(wl, want_scores=True)
    check_sparse_step(eng, wl)
    eng.dense_decode()
    torch.cuda.synchronize()
    check_dense(eng, wl)


def test_many_short_sequences():
    """700 sequences, most of them a few pages long: more sequences than the decode CTA has threads (its prefix table is then
    built several sequences per thread), units far smaller than a CTA's piece (tens of parts per CTA), many empty slices in
    the selector's grid, sequences that go dense inside the sparse batch."""
    rng = np.random.default_rng(11)
    lens = [int(x) for x in rng.integers(1, 700, size=700)]
    lens[5], lens[77], lens[699] = 1, 16, 2500
    sched = W._sched("fixed", 16, 32, fixed_tokens=96)
    wl = W.make_workload(n_seq=len(lens), Hq=4, Hkv=2, lengths=("list", lens), schedule=sched, seed=4242, device=DEV, poison_tail=True, plant=True)
    eng = _run_sparse(wl, want_scores=True)
    check_sparse_step(eng, wl)
    eng.dense_decode()
    torch.cuda.synchronize()
    check_dense(eng, wl)


@pytest.mark.parametrize("Hq,Hkv,page,landmark", [(8, 2, 16, "minmax"), (5, 1, 16, "minmax"), (16, 8, 64, "minmax"), (8, 2, 32, "mean")])
def test_strided_nhd_pools_match_the_oracle_and_the_packed_layout(Hq, Hkv, page, landmark):
    """sparrow_shape_t kv_stride_*: the same K/V values in pools laid out [page][token][kv-head][128] (NHD, the default of
    vLLM / FlashInfer) go through summarize, select, decode (5-D TMA boxes), the dense entry and append; everything is
    checked against the oracle (which sees the packed arrays) and the appended caches against the packed run's, bit for bit."""
    import copy
    from paper_2606_08446_b200.engine import SparrowEngine
    lens = [1, 16, 17, 250, 1000, 2049, 4099, 700]
    sched = W._sched("fixed", 16, 64, fixed_tokens=300)
    wl = W.make_workload(n_seq=len(lens), Hq=Hq, Hkv=Hkv, lengths=("list", lens), schedule=sched, seed=Hq * 31 + page, device=DEV,
                         poison_tail=True, plant=True, page_size=page, reserve_tokens=8)
    nhd = copy.copy(wl)
    nhd.k_cache = wl.k_cache.permute(0, 2, 1, 3).contiguous()          # [n_phys][P][Hkv][128]
    nhd.v_cache = wl.v_cache.permute(0, 2, 1, 3).contiguous()
    nhd.seq_lens = wl.seq_lens.clone()
    eng = SparrowEngine(nhd, want_scores=(landmark == "minmax"), landmark=landmark, kv_layout="nhd")
    ref = SparrowEngine(wl, landmark=landmark)
    for e in (eng, ref):
        e.summarize_all(); e.step(); e.dense_decode()
    torch.cuda.synchronize()
    assert torch.equal(eng.summaries, ref.summaries) and torch.equal(eng.sel_pages, ref.sel_pages) and torch.equal(eng.sel_count, ref.sel_count)
    if landmark == "minmax":
        check_sparse_step(eng, wl)
        check_dense(eng, wl)
    assert_same_result(eng.out, ref.out, "NHD vs packed", eng.lse, ref.lse)
    assert_same_result(eng.out_dense, ref.out_dense, "NHD vs packed, dense entry", eng.lse_dense, ref.lse_dense)
    # rollout side: four appended tokens per sequence land in the same logical rows, and pages that fill get the same summaries
    for e in (eng, ref):
        e.reserve(4)
    qs, ks, vs = W.make_rollout_inputs(wl, 4, seed=9)
    for t in range(4):
        eng.append(ks[t], vs[t]); ref.append(ks[t], vs[t])
    torch.cuda.synchronize()
    assert torch.equal(nhd.k_cache.permute(0, 2, 1, 3), wl.k_cache) and torch.equal(nhd.v_cache.permute(0, 2, 1, 3), wl.v_cache)
    assert torch.equal(eng.summaries, ref.summaries) and torch.equal(nhd.seq_lens, wl.seq_lens)


@pytest.mark.parametrize("page", [16, 64])
def test_non_finite_bits_in_unwritten_tails_never_reach_the_output(page):
    """A torch.empty pool or a recycled page leaves arbitrary bit patterns in the rows past L of a sequence's last page
    (and, for pages larger than 16 tokens, in whole 16-token sub-tiles past L).  The oracle never reads them; neither
    may the kernels: K tails = NaN, V tails = +Inf here (0 x Inf in the P V product would be NaN)."""
    lens = [1, 15, 17, 33, page + 1, 250, 257, 1000, 2049, 4099]
    sched = W._sched("fixed", 16, 64, fixed_tokens=320)
    wl = W.make_workload(n_seq=len(lens), Hq=8, Hkv=2, lengths=("list", lens), schedule=sched, seed=31 + page, device=DEV,
                         poison_tail="nonfinite", plant=True, page_size=page)
    assert not torch.isfinite(wl.k_cache.float()).all() and not torch.isfinite(wl.v_cache.float()).all()
    eng = _run_sparse(wl, want_scores=True)
    check_sparse_step(eng, wl)
    eng.dense_decode()
    torch.cuda.synchronize()
    check_dense(eng, wl)


@pytest.mark.parametrize("sched", [
    W._sched("clamp_frac", 64, 512, f0_ppm=125000, floor_tokens=2048),
    W._sched("linear_frac", 64, 512, f0_ppm=250000, f1_ppm=62500, L0=8192, L1=32768, floor_tokens=2048),
    W._sched("clamp_frac", 0, 0, f0_ppm=50000, floor_tokens=64),
    W._sched("table", 32, 100, table_pages=(8, 20, 40, 50, 64, 70), bin_tokens=2048),
    W._sched("fixed", 700, 900, fixed_tokens=64),      # forced pages exceed the budget: k = 0 (R2)
    W._sched("dense", 0, 0),
], ids=["cfg2-clamp", "cfg3-linear", "nosink-nolocal", "table-2k-bins", "forced-exceed-budget", "dense-kind"])
def test_schedules_medium_batch(sched):
    # lengths span one to ~44 select chunks (256 pages) and many decode splits, with ragged tails
    lens = [300, 2047, 2048, 2049, 4096, 5000, 8191, 9001, 11111, 700, 16, 6143]
    wl = W.make_workload(n_seq=len(lens), Hq=8, Hkv=2, lengths=("list", lens), schedule=sched, seed=77, device=DEV, plant=True)
    eng = _run_sparse(wl, want_scores=True)
    check_sparse_step(eng, wl)


def test_near_tie_across_the_threshold_takes_the_band_and_r11_path():
    """R10 / R11 on GPU data.  Per unit, the page at the top-k threshold (A) is copied onto an unselected candidate with a
    HIGHER index (B), and one key of B is raised by one bf16 step in a channel where the group's queries are 2^-20: in
    fp64 B now outscores A by ~1e-8 (relative 1e-11, far inside the 1e-4 band) and the oracle picks B; in fp32 the two
    scores round to the same number and the kernel's tie rule keeps A.  Both are valid results: the checker must accept the
    list through the band rule and compare the attention on the GPU's own sets -- branches no other test has reached."""
    lens = [3000, 4100, 2500, 5000]
    wl = W.make_workload(n_seq=len(lens), Hq=8, Hkv=2, lengths=("list", lens), schedule=W._sched("fixed", 64, 256, fixed_tokens=1024),
                         seed=91, device=DEV, plant=True)
    d0 = 5
    wl.q[:, :, d0] = 2.0 ** -20
    h = wl.host()
    sched = oracle.Schedule.from_spec(wl.schedule)
    res = oracle.sparse_step(h["q"], h["k_cache"], h["v_cache"], h["page_table"], h["seq_lens"], sched, wl.sm_scale, do_attention=False)
    made = 0
    for i, L in enumerate(lens):
        n_pages = -(-L // 16)
        F = set(np.flatnonzero(res["forced"][i, :n_pages]).tolist())
        cnt = int(res["sel_count"][i])
        for g in range(wl.Hkv):
            row = set(res["sel"][i, g, :cnt].tolist())
            top = sorted(row - F, key=lambda p: res["scores"][i, g, p])
            a = top[0]                                                # the page at the threshold
            assert res["scores"][i, g, a] == res["tau"][i, g] and res["scores"][i, g, top[1]] > res["tau"][i, g]
            b = max(p for p in range(n_pages) if p not in row and p > a)
            pa, pb = int(wl.page_table[i, a]), int(wl.page_table[i, b])
            wl.k_cache[pb, g] = wl.k_cache[pa, g]
            col = wl.k_cache[pb, g, :, d0]
            t = int(col.float().argmax())
            bits = col.view(torch.int16)
            assert float(col[t]) != 0.0
            bits[t] += 1 if float(col[t]) > 0 else -1                # one bf16 step up: the page's max in channel d0 rises
            made += 1
    eng = _run_sparse(wl, want_scores=True)
    st = check_sparse_step(eng, wl)
    print(f"near ties planted in {made} units: {st}")
    assert st["differing_units"] >= made // 2 and st["band_pages"] >= 2 * (made // 2)


def test_all_ties_zero_query_picks_lowest_pages():
    lens = [1200, 640, 5000]
    sched = W._sched("fixed", 16, 32, fixed_tokens=320)
    wl = W.make_workload(n_seq=3, Hq=4, Hkv=2, lengths=("list", lens), schedule=sched, seed=5, device=DEV)
    wl.q.zero_()
    eng = _run_sparse(wl)
    st = check_sparse_step(eng, wl)
    assert st["differing_units"] == 0       # exact ties resolve to the lower page index on both sides
    assert eng.sel_pages[0, 0, :20].tolist() == list(range(18)) + [73, 74]   # F = {0, 73, 74}, k = 17


def test_summarize_bulk_identity_and_partial_pages():
    from paper_2606_08446_b200.engine import SparrowEngine
    wl = W.make_workload(n_seq=3, Hq=4, Hkv=4, lengths=("list", [100, 37, 513]), schedule=W._sched("dense", 0, 0), seed=9, device=DEV)
    h = wl.host()
    eng = SparrowEngine(wl)
    eng.summarize(None, None, n_update=wl.n_phys)            # page_ids = NULL: pages 0..n-1, all 16 tokens
    torch.cuda.synchronize()
    check_summaries(eng.summaries, h, np.arange(wl.n_phys), None)
    ids = torch.tensor([5, 0, 7], dtype=torch.int32, device=DEV)
    nv = torch.tensor([1, 9, 16], dtype=torch.int32, device=DEV)
    eng.summarize(ids, nv)
    torch.cuda.synchronize()
    check_summaries(eng.summaries, h, ids.cpu().numpy(), nv.cpu().numpy())


def test_select_is_repeatable_and_graph_capturable():
    wl = W.make_workload(n_seq=6, Hq=8, Hkv=4, lengths=("list", [3000, 4000, 513, 9000, 77, 2500]),
                         schedule=W._sched("fixed", 64, 256, fixed_tokens=1024), seed=3, device=DEV, plant=True)
    eng = _run_sparse(wl)
    ref_sel, ref_out = eng.sel_pages.clone(), eng.out.clone()
    st = torch.cuda.Stream()
    with torch.cuda.stream(st):
        eng.sel_pages.fill_(-1); eng.out.zero_()
        eng.step(stream=st)                                   # warm-up on the capture stream
        st.synchronize()
        g = torch.cuda.CUDAGraph()
        with torch.cuda.graph(g, stream=st):
            eng.step(stream=st)
        for _ in range(3):
            eng.sel_pages.fill_(-1); eng.out.zero_()
            g.replay()
    st.synchronize()
    torch.cuda.synchronize()
    assert torch.equal(eng.sel_pages, ref_sel)                 # the selection is exact and reproducible
    assert_same_result(eng.out, ref_out, "graph replay")      # the attention to within the arithmetic's error (run-time tile hand-out)
    check_sparse_step(eng, wl)


def test_step_host_entry_matches_device_path():
    from paper_2606_08446_b200 import binding as B
    wl = W.make_workload(n_seq=5, Hq=8, Hkv=2, lengths=("list", [2048, 4000, 160, 3333, 4096]),
                         schedule=W._sched("clamp_frac", 64, 256, f0_ppm=125000, floor_tokens=512), seed=13, device=DEV, plant=True)
    eng = _run_sparse(wl)
    ids, nv = W.just_filled_updates(wl)
    assert ids.numel() == 4
    scratch = torch.zeros((B.sparrow_step_scratch_bytes(eng.shape, eng.max_sel),), dtype=torch.uint8, device=DEV)
    hb = B.HostBlock(eng.shape)                               # one pinned block: q | seq_lens | page_ids | n_valid
    hb.q.copy_(wl.q.cpu()); hb.seq_lens.copy_(wl.seq_lens.cpu())
    hb.page_ids[: ids.numel()] = ids; hb.n_valid[: ids.numel()] = nv
    out_h = torch.zeros_like(hb.q).pin_memory()
    eng.summaries[ids.long().to(DEV)] = 0                     # the step must rebuild the summaries of just-filled pages
    B.sparrow_step_host(hb.block, ids.numel(), True, wl.k_cache, wl.v_cache, eng.summaries, wl.page_table,
                        eng.sched, eng.max_sel, wl.sm_scale, out_h, scratch, eng.shape)
    assert B.sparrow_last_launch_count() == 3                 # summarize, select, decode (merge fused in the decode launch)
    assert_same_result(out_h, eng.out.cpu(), "host-buffer entry vs device path")
    check_summaries(eng.summaries, wl.host(), ids.numpy(), nv.numpy())


def test_error_statuses_on_device_calls():
    from paper_2606_08446_b200 import binding as B
    wl = W.make_config("cfg1", device=DEV)
    eng = _engine(wl)
    small = torch.empty((16,), dtype=torch.uint8, device=DEV)
    rc = B.sparrow_sparse_decode(wl.q, wl.k_cache, wl.v_cache, wl.page_table, wl.seq_lens, eng.sel_pages, eng.max_sel,
                                 eng.sel_count, eng.out, eng.lse, wl.sm_scale, small, eng.shape, check=False)
    assert rc == -3
    q_mis = torch.empty((wl.q.numel() + 8,), dtype=torch.bfloat16, device=DEV)[1:1 + wl.q.numel()].view_as(wl.q)
    assert q_mis.is_contiguous() and q_mis.data_ptr() % 16 != 0
    rc = B.sparrow_select(q_mis, eng.summaries, wl.page_table, wl.seq_lens, eng.sched, eng.sel_pages, eng.max_sel,
                          eng.sel_count, None, eng.select_ws, eng.shape, check=False)
    assert rc == -1                                            # misaligned device pointer
    with pytest.raises(B.SparrowError):
        B.sparrow_dense_decode(wl.q, wl.k_cache, wl.v_cache, wl.page_table, wl.seq_lens, eng.out_dense, eng.lse_dense,
                               wl.sm_scale, small, eng.shape)


# ------------------------------------------------------------------ full-size BASELINE.json configs ----
# The launch configuration bench.py times.  Selection (count, order, range, F, band rule, fp32 scores) and the summaries
# are checked on EVERY sequence of the batch, and so are out / lse (the oracle needs about a second per config on the box's
# cores; the n_out parameter remains for sampling, unused).  The dense entry is compared on the shortest and the longest
# sequence and on sequences of cfg4 that go dense inside the sparse batch.
@pytest.mark.parametrize("cfg,n_out", [("cfg2", None), ("cfg5", None), ("cfg3", None), ("cfg4", None)])
def test_full_size_config_against_oracle(cfg, n_out):
    wl = W.make_config(cfg, device=DEV)
    eng = _run_sparse(wl, want_scores=True)
    eng.dense_decode()                   # cfg4: the call its layers 0-1 make
    torch.cuda.synchronize()
    h = wl.host()
    lens = h["seq_lens"]
    sched = oracle.Schedule.from_spec(wl.schedule)
    if n_out is None:
        out_idx = None
        dense_idx = sorted({int(lens.argmin()), int(lens.argmax()), 1})
    else:
        rng = np.random.default_rng(1)
        dense_inside = [i for i in range(wl.n_seq) if oracle.k_pages(sched, int(lens[i])) >= -(-int(lens[i]) // 16)]
        must = sorted(set([int(lens.argmin()), int(lens.argmax())] + dense_inside[:8]))
        rest = [i for i in rng.permutation(wl.n_seq).tolist() if i not in must]
        out_idx = sorted(must + rest[: n_out - len(must)])
        dense_idx = sorted(set([int(lens.argmin()), int(lens.argmax())] + dense_inside[:2]))
        if cfg == "cfg4":                # log-normal lengths: short sequences go dense inside the sparse batch
            assert int(lens.min()) < 2048 and len(dense_inside) >= 1
    st = check_sparse_step(eng, wl, h=h, out_idx=out_idx)
    sd = check_dense(eng, wl, h=h, idx=dense_idx)
    print(f"{cfg}: {st}; dense on {dense_idx}: {sd}")
    assert st["seqs_selection"] == wl.n_seq and st["seqs_outputs"] == (wl.n_seq if n_out is None else n_out)
    assert torch.isfinite(eng.out.float()).all() and torch.isfinite(eng.lse).all()
    # planted pages that are candidates are (almost all) recovered: the selector is meaningful on this workload
    cnt = eng.sel_count.cpu().numpy()
    sel = eng.sel_pages.cpu().numpy()
    rec, tot = 0, 0
    for i in range(wl.n_seq):
        L = int(lens[i])
        F = set(np.flatnonzero(oracle.forced_pages(L, sched.sink_tokens, sched.local_tokens)).tolist())
        k = cnt[i] - len(F)
        for g in range(wl.Hkv):
            row = set(sel[i, g, :cnt[i]].tolist())
            pl = [p for p in wl.planted[i][g].tolist() if p not in F]
            rec += sum(p in row for p in pl); tot += min(len(pl), k)
    print(f"{cfg}: planted candidates recovered {rec}/{tot}")
    assert rec >= 0.8 * tot


# ------------------------------------------------------------------ 8(f)-2: page sizes 32 / 64 / 128 ----
@pytest.mark.parametrize("page", [32, 64, 128])
@pytest.mark.parametrize("Hq,Hkv", [(8, 2), (5, 1)])
def test_page_size_variants_match_oracle(page, Hq, Hkv):
    """Table 4's page sizes: a page is streamed as page/16 tiles; summaries, selection, sparse and
    dense attention against the oracle at that page size; ragged lengths around tile and page edges."""
    lens = [1, 15, 16, 17, page - 1, page, page + 1, 3 * page + 5, 1000, 2049, 4099, 6000]
    sched = W._sched("fixed", 16, 64, fixed_tokens=1024)          # Table 4's budget 1024: 32-32, 64-16, 128-8
    wl = W.make_workload(n_seq=len(lens), Hq=Hq, Hkv=Hkv, lengths=("list", lens), schedule=sched, seed=page + Hq, device=DEV,
                         poison_tail=True, plant=True, page_size=page)
    eng = _run_sparse(wl, want_scores=True)
    st = check_sparse_step(eng, wl)
    assert eng.sel_count.cpu().tolist() == [min(-(-L // page), max(1024 // page, len(set([0]) | set(range(max(L - 64, 0) // page, -(-L // page)))))) for L in lens]
    eng.dense_decode()
    torch.cuda.synchronize()
    check_dense(eng, wl)


def test_rollout_with_page_size_64():
    """append + summarize-on-fill + select + decode at page size 64: 70 steps cross a page edge for every sequence."""
    from paper_2606_08446_b200.engine import SparrowEngine
    T, lens = 70, [100, 1000, 4000]
    sched = W._sched("clamp_frac", 64, 128, f0_ppm=250000, floor_tokens=512)
    wl = W.make_workload(n_seq=3, Hq=8, Hkv=2, lengths=("list", lens), schedule=sched, seed=64, device=DEV, plant=True,
                         page_size=64, reserve_tokens=T + 1)
    eng = SparrowEngine(wl, want_scores=True)
    eng.summarize_all(); eng.reserve(T)
    qs, ks, vs = W.make_rollout_inputs(wl, T, seed=9)
    bits = lambda t: t.contiguous().view(torch.int16).cpu().numpy().view(np.uint16)
    h0 = wl.host()
    want, kc, vc = oracle.rollout(bits(qs), bits(ks), bits(vs), h0["k_cache"], h0["v_cache"], h0["page_table"], h0["seq_lens"],
                                  oracle.Schedule.from_spec(sched), wl.sm_scale, max_sel=eng.max_sel)
    out = torch.zeros((T, 3, 8, 128), dtype=torch.bfloat16, device=DEV)
    lse = torch.zeros((T, 3, 8), dtype=torch.float32, device=DEV)
    # three segments, so that the page lists of steps 0, T/2 and T-1 can be read back and checked
    from parity_util import check_selection
    checked = {}
    for a, b in ((0, 1), (1, T // 2 + 1), (T // 2 + 1, T)):
        eng.rollout(qs[a:b], ks[a:b], vs[a:b], out[a:b], lse[a:b])
        torch.cuda.synchronize()
        checked[b - 1] = (eng.sel_pages.cpu().numpy().copy(), eng.sel_count.cpu().numpy().copy(), eng.scores.cpu().numpy().copy())
    assert np.array_equal(bits(wl.k_cache), kc) and np.array_equal(bits(wl.v_cache), vc)
    filled = sorted(p for s in want for p in s["filled"])
    assert len(filled) >= 3
    check_summaries(eng.summaries, dict(k_cache=kc), np.array(filled), None)
    # every checked step: selection by the band rule, then out / lse against the oracle's attention on the GPU's own
    # validated sets (R11) -- unconditionally.  Tokens below L_t never change after step t, so the final cache with
    # step t's lengths is the cache of step t.
    for t, (sel_gpu, cnt_gpu, sc_gpu) in checked.items():
        check_selection(want[t], sel_gpu, cnt_gpu, want[t]["seq_lens"], sc_gpu, page_size=64)
        sel_fix = np.where(np.arange(sel_gpu.shape[2])[None, None, :] < cnt_gpu[:, None, None], sel_gpu, 0)
        w_out, w_lse = oracle.attention_on_sets(bits(qs[t]), kc, vc, h0["page_table"], want[t]["seq_lens"], np.ascontiguousarray(sel_fix),
                                                cnt_gpu.astype(np.int64), wl.sm_scale)
        check_outputs(out[t], lse[t], w_out, w_lse, f"page-64 rollout step {t}")


# ------------------------------------------------------------------ 8(f)-2: the mean-key landmark ----
@pytest.mark.parametrize("Hq,Hkv,page", [(8, 2, 16), (5, 1, 16), (16, 8, 16), (8, 2, 64)])
def test_mean_landmark_matches_oracle(Hq, Hkv, page):
    """One vector per page (the paper's cost model): landmarks == the exact mean rounded once to bf16, or its
    neighbour inside the fp32-accumulation band (R24); scores, selection (band rule) and attention against oracle.sparse_step_mean; ragged lengths, partial pages."""
    lens = [1, 15, 16, 17, 33, 250, 256, 257, 1000, 2049, 4099, 9000]
    sched = W._sched("fixed", 16, 64, fixed_tokens=320)
    wl = W.make_workload(n_seq=len(lens), Hq=Hq, Hkv=Hkv, lengths=("list", lens), schedule=sched, seed=Hq * 10 + page, device=DEV,
                         poison_tail=True, plant=True, page_size=page)
    eng = _run_sparse(wl, want_scores=True, landmark="mean")
    assert eng.summaries.shape == (wl.n_phys, Hkv, 128)
    check_sparse_step(eng, wl)


def test_mean_landmark_rollout_summarizes_on_fill():
    from paper_2606_08446_b200.engine import SparrowEngine
    T, lens = 40, [100, 1000, 4090]
    sched = W._sched("clamp_frac", 32, 96, f0_ppm=125000, floor_tokens=256)
    wl = W.make_workload(n_seq=3, Hq=8, Hkv=2, lengths=("list", lens), schedule=sched, seed=8, device=DEV, plant=True, reserve_tokens=T + 1)
    eng = SparrowEngine(wl, want_scores=True, landmark="mean")
    eng.summarize_all(); eng.reserve(T)
    qs, ks, vs = W.make_rollout_inputs(wl, T, seed=2)
    out = torch.zeros((T, 3, 8, 128), dtype=torch.bfloat16, device=DEV)
    eng.rollout(qs, ks, vs, out)
    torch.cuda.synchronize()
    # after the rollout the engine state is a plain step on the grown cache: landmarks (incl. pages filled on the way),
    # selection and the last step's attention all checked against the oracle on the final cache
    wl.q = qs[T - 1].contiguous()
    eng.out.copy_(out[T - 1])
    eng.sparse_decode(wl.q)                                          # refresh lse for the checker
    torch.cuda.synchronize()
    assert wl.seq_lens.cpu().tolist() == [L + T for L in lens]
    h = wl.host()
    ids = np.concatenate([h["page_table"][i, :(L + T) // 16] for i, L in enumerate(lens)])      # every FULL page
    check_summaries(eng.summaries, h, ids, None)
    check_sparse_step(eng, wl, h=h, check_summ=False)
