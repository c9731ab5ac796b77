"""SPARROW_FLAG_DETERMINISTIC (``-m gpu``): with the flag the decode's tile hand-out and merge orders are fixed, so two
calls on the same inputs must agree BIT FOR BIT -- out, lse, and of course the page lists -- and the result must still pass
the oracle's gates.  This is the bitwise guard the run-time hand-out of the default mode cannot give (tests there use
parity_util.assert_same_result, a tolerance); the protocol that could drop or double-count a small partial -- parking areas,
cross-piece partials, the completing part's fast path -- is the same code in both modes, so an intermittent slip in it shows
here as a differing bit instead of hiding inside a tolerance.  PAPER.md:76-79, :409-414: the paper's subject is the
log-prob mismatch between rollout and trainer; a rollout kernel should not add a source of its own."""
import pytest
import torch

from paper_2606_08446_b200 import workloads as W

from parity_util import check_dense, check_sparse_step

pytestmark = pytest.mark.gpu
DEV = "cuda"


def _engine(wl, **kw):
    from paper_2606_08446_b200.engine import SparrowEngine
    eng = SparrowEngine(wl, deterministic=True, **kw)
    eng.summarize_all()
    return eng


def _repeat_bitwise(eng, n_runs, dense_runs=0):
    eng.step()
    torch.cuda.synchronize()
    sel0, cnt0, out0, lse0 = eng.sel_pages.clone(), eng.sel_count.clone(), eng.out.clone(), eng.lse.clone()
    for i in range(n_runs):
        eng.sel_pages.fill_(-1); eng.sel_count.zero_(); eng.out.zero_(); eng.lse.zero_()
        eng.step()
        torch.cuda.synchronize()
        assert torch.equal(eng.sel_pages, sel0) and torch.equal(eng.sel_count, cnt0), f"run {i}: selection differs"
        assert torch.equal(eng.out, out0), f"run {i}: out differs in {(eng.out != out0).sum().item()} elements"
        assert torch.equal(eng.lse, lse0), f"run {i}: lse differs"
    if dense_runs:
        eng.dense_decode()
        torch.cuda.synchronize()
        d0, l0 = eng.out_dense.clone(), eng.lse_dense.clone()
        for i in range(dense_runs):
            eng.out_dense.zero_(); eng.lse_dense.zero_()
            eng.dense_decode()
            torch.cuda.synchronize()
            assert torch.equal(eng.out_dense, d0) and torch.equal(eng.lse_dense, l0), f"dense run {i} differs"


@pytest.mark.parametrize("cfg", ["cfg2", "cfg5"])
def test_full_size_step_is_bit_reproducible(cfg):
    """The launch configuration bench.py times, 20 times over: every unit spans parts of several consumers, most CTAs end
    inside a unit (cross-piece partials, both the completing part's fast path and the slow path occur)."""
    wl = W.make_config(cfg, device=DEV)
    eng = _engine(wl)
    _repeat_bitwise(eng, 20, dense_runs=3)
    check_sparse_step(eng, wl, check_summ=False, out_idx=list(range(0, wl.n_seq, 4)))      # and it is still the right answer


@pytest.mark.parametrize("Hq,Hkv,page,lens,budget", [
    (8, 2, 16, [33000], 9000),                      # one unit per kv-head over tens of CTAs: up to 74 partials per unit
    (5, 1, 16, [20000, 17, 3, 9000], 6000),         # r = 5, tiny units between long ones
    (16, 8, 64, [40000, 300, 25000], 20000),        # page 64: four tiles per page
    (2, 2, 16, [1, 15, 16, 17, 33, 250, 256, 257, 1000, 2049, 4099], 200),   # r = 1, ragged
])
def test_bit_reproducible_and_oracle_exact_on_awkward_shapes(Hq, Hkv, page, lens, budget):
    sched = W._sched("fixed", 16, 64, fixed_tokens=budget)
    wl = W.make_workload(n_seq=len(lens), Hq=Hq, Hkv=Hkv, lengths=("list", lens), schedule=sched, seed=Hq * 7 + Hkv, device=DEV,
                         plant=True, poison_tail=True, page_size=page)
    eng = _engine(wl, want_scores=True)
    _repeat_bitwise(eng, 10, dense_runs=5)
    check_sparse_step(eng, wl)
    check_dense(eng, wl)


def test_many_short_sequences_bit_reproducible():
    """The workload of test_gpu_parity.test_many_short_sequences: tens of parts per CTA, more sequences than decode threads."""
    import numpy as np
    rng = np.random.default_rng(11)
    lens = [int(x) for x in rng.integers(1, 700, size=700)]
    lens[5], lens[77], lens[699] = 1, 16, 2500
    wl = W.make_workload(n_seq=len(lens), Hq=4, Hkv=2, lengths=("list", lens), schedule=W._sched("fixed", 16, 32, fixed_tokens=96),
                         seed=4242, device=DEV, poison_tail=True, plant=True)
    eng = _engine(wl, want_scores=True)
    _repeat_bitwise(eng, 10, dense_runs=5)
    check_sparse_step(eng, wl)
    check_dense(eng, wl)


def test_graph_replay_and_host_entry_are_bitwise_equal_to_the_eager_device_path():
    from paper_2606_08446_b200 import binding as B
    wl = W.make_workload(n_seq=6, Hq=8, Hkv=4, lengths=("list", [3000, 4000, 513, 9000, 77, 2500]),
                         schedule=W._sched("fixed", 64, 256, fixed_tokens=1024), seed=3, device=DEV, plant=True)
    eng = _engine(wl)
    eng.step()
    torch.cuda.synchronize()
    ref_sel, ref_out, ref_lse = eng.sel_pages.clone(), eng.out.clone(), eng.lse.clone()
    st = torch.cuda.Stream()
    with torch.cuda.stream(st):
        eng.step(stream=st)
        st.synchronize()
        g = torch.cuda.CUDAGraph()
        with torch.cuda.graph(g, stream=st):
            eng.step(stream=st)
        for _ in range(5):
            eng.sel_pages.fill_(-1); eng.out.zero_(); eng.lse.zero_()
            g.replay()
            st.synchronize()
            assert torch.equal(eng.sel_pages, ref_sel) and torch.equal(eng.out, ref_out) and torch.equal(eng.lse, ref_lse)
    torch.cuda.synchronize()
    # the host-buffer entry runs the same kernels on its own scratch: same bits
    scratch = torch.zeros((B.sparrow_step_scratch_bytes(eng.shape, eng.max_sel),), dtype=torch.uint8, device=DEV)
    hb = B.HostBlock(eng.shape)
    hb.q.copy_(wl.q.cpu()); hb.seq_lens.copy_(wl.seq_lens.cpu())
    out_h = torch.zeros_like(hb.q).pin_memory()
    B.sparrow_step_host(hb.block, 0, False, wl.k_cache, wl.v_cache, eng.summaries, wl.page_table, eng.sched, eng.max_sel,
                        wl.sm_scale, out_h, scratch, eng.shape)
    assert torch.equal(out_h, ref_out.cpu())
    # ... and so does the enqueue-only form, several steps in flight on one stream sharing the scratch, one wait at the end
    outs = [torch.zeros_like(hb.q).pin_memory() for _ in range(4)]
    for o in outs:
        B.sparrow_step_host(hb.block, 0, False, wl.k_cache, wl.v_cache, eng.summaries, wl.page_table, eng.sched, eng.max_sel,
                            wl.sm_scale, o, scratch, eng.shape, wait=False)
    torch.cuda.current_stream().synchronize()
    for o in outs:
        assert torch.equal(o, ref_out.cpu())


def test_unknown_flag_bits_are_refused():
    from paper_2606_08446_b200 import binding as B
    shp = B.make_shape(2, 4, 2, 8, 16)
    assert B.sparrow_decode_workspace_bytes(shp, 4) > 0
    shp.flags = 2
    assert B.sparrow_decode_workspace_bytes(shp, 4) == 0      # check_shape: INVALID_ARG
    shp.flags = B.FLAG_DETERMINISTIC
    assert B.sparrow_decode_workspace_bytes(shp, 4) > 0


def test_rollout_as_one_graph_is_bitwise_equal_to_step_by_step():
    """The rollout chain append -> select -> decode, T steps: run step by step and as ONE CUDA graph on a fresh copy of the
    batch.  With the flag the two must agree in every bit of every step's out and lse (the default mode's version of this
    check, tests/test_gpu_rollout.py, can only assert a tolerance)."""
    from paper_2606_08446_b200.engine import SparrowEngine
    T, lens = 20, [250, 1023, 15, 2040, 4090]
    sched = W._sched("table", 16, 48, table_pages=(6, 9, 14, 20, 20, 24, 24, 30, 40), bin_tokens=512)

    def setup():
        wl = W.make_workload(n_seq=len(lens), Hq=8, Hkv=2, lengths=("list", lens), schedule=sched, seed=21, device=DEV,
                             reserve_tokens=T + 3, plant=True)
        eng = SparrowEngine(wl, deterministic=True)
        eng.summarize_all()
        eng.reserve(T)
        return (wl, eng) + tuple(W.make_rollout_inputs(wl, T, seed=5))

    wl, eng, qs, ks, vs = setup()
    out = torch.zeros((T, wl.n_seq, wl.Hq, 128), dtype=torch.bfloat16, device=DEV)
    lse = torch.zeros((T, wl.n_seq, wl.Hq), dtype=torch.float32, device=DEV)
    for t in range(T):
        eng.append(ks[t], vs[t]); eng.select(qs[t]); eng.sparse_decode(qs[t], out=out[t], lse=lse[t])
        torch.cuda.synchronize()
    wl2, eng2, qs2, ks2, vs2 = setup()
    out2, lse2 = torch.zeros_like(out), torch.zeros_like(lse)
    st = torch.cuda.Stream()
    with torch.cuda.stream(st):
        g = torch.cuda.CUDAGraph()
        with torch.cuda.graph(g, stream=st):
            eng2.rollout(qs2, ks2, vs2, out2, lse2, stream=st)
        g.replay()
    st.synchronize()
    torch.cuda.synchronize()
    assert wl2.seq_lens.cpu().tolist() == [L + T for L in lens]
    assert torch.equal(out2, out) and torch.equal(lse2, lse)
    assert torch.equal(wl2.k_cache, wl.k_cache) and torch.equal(eng2.summaries, eng.summaries)


@pytest.mark.parametrize("Hq,Hkv,page", [(8, 2, 16), (5, 1, 16), (16, 8, 64)])
def test_nhd_pools_give_the_same_bits_as_packed_pools(Hq, Hkv, page):
    """Strided pools are fetched with 5-D TMA boxes that land in shared memory exactly as the packed layout's 2-D boxes do:
    same tiles, same hand-out, so -- with the flag -- the same bits out of the sparse and the dense entry."""
    import copy
    from paper_2606_08446_b200.engine import SparrowEngine
    lens = [1, 16, 17, 250, 1000, 2049, 4099, 700]
    wl = W.make_workload(n_seq=len(lens), Hq=Hq, Hkv=Hkv, lengths=("list", lens), schedule=W._sched("fixed", 16, 64, fixed_tokens=300),
                         seed=Hq * 31 + page, device=DEV, poison_tail=True, plant=True, page_size=page)
    nhd = copy.copy(wl)
    nhd.k_cache = wl.k_cache.permute(0, 2, 1, 3).contiguous()
    nhd.v_cache = wl.v_cache.permute(0, 2, 1, 3).contiguous()
    eng = SparrowEngine(nhd, kv_layout="nhd", deterministic=True)
    ref = SparrowEngine(wl, deterministic=True)
    for e in (eng, ref):
        e.summarize_all(); e.step(); e.dense_decode()
    torch.cuda.synchronize()
    assert torch.equal(eng.sel_pages, ref.sel_pages) and torch.equal(eng.sel_count, ref.sel_count)
    assert torch.equal(eng.out, ref.out) and torch.equal(eng.lse, ref.lse)
    assert torch.equal(eng.out_dense, ref.out_dense) and torch.equal(eng.lse_dense, ref.lse_dense)
    check_sparse_step(ref, wl, check_summ=False)
