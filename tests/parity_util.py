"""Checker shared by the GPU parity tests, smoke() and the bench's self-check (SURVEY.md section 8(c) procedure).

Compares what the CUDA library produced with the fp64 oracle on the same bit patterns:
  (1) summaries: numeric equality; (2) selection: same count, ascending, in range, contains F, symmetric
  difference only inside the tie band |s - tau| <= 1e-4 |tau| (north_star; oracle fp64 scores);
  (3) out / lse against the oracle evaluated on the GPU's own page sets (R11; identical to the oracle's own
  result when the sets agree), with north_star's tolerances and the tighter internal gates.
"""
from __future__ import annotations

import numpy as np
import torch

import oracle

# north_star: bf16 outputs, fp32 accumulation
TOL_MAX_ABS = 2e-2
TOL_MEAN_ABS = 2e-3
# tighter internal gates: catch a dropped / duplicated page
# elementwise |err| <= GATE_ABS + GATE_REL*|want|: bf16 output rounding is 2^-9 |out|, bf16 P adds ~2^-9 * sqrt(sum p^2) * |v|
GATE_ABS = 2e-3
GATE_REL = 2.0 ** -8
GATE_MEAN_ABS = 3e-4
GATE_LSE_ABS = 1e-3
BAND_REL = 1e-4


def bf16_to_f64(t: torch.Tensor) -> np.ndarray:
    return t.detach().float().cpu().numpy().astype(np.float64)


def sub_host(h: dict, idx) -> dict:
    """Host view of a subset of sequences (the K/V pools stay whole).  `h` is Workload.host() or a
    workloads.host_subset() view; idx are ORIGINAL sequence numbers."""
    idx = np.asarray(idx)
    if "seq_index" in h:                     # compacted view: rows are h["seq_index"]
        where = {int(s): j for j, s in enumerate(h["seq_index"].tolist())}
        idx = np.array([where[int(s)] for s in idx], dtype=np.int64)
    return dict(q=np.ascontiguousarray(h["q"][idx]), k_cache=h["k_cache"], v_cache=h["v_cache"],
                page_table=np.ascontiguousarray(h["page_table"][idx]), seq_lens=np.ascontiguousarray(h["seq_lens"][idx]),
                phys_ids=h.get("phys_ids"))


def _gpu_rows(summ_gpu: torch.Tensor, h: dict, page_ids) -> torch.Tensor:
    """Rows of the GPU's summaries for host pages `page_ids` (renumbered back when `h` is a compacted view)."""
    ids = np.asarray(page_ids)
    if h.get("phys_ids") is not None:
        ids = np.asarray(h["phys_ids"])[ids]
    return summ_gpu[torch.as_tensor(ids).long().to(summ_gpu.device)]


def check_summaries(summ_gpu: torch.Tensor, h: dict, page_ids, n_valid):
    if summ_gpu.dim() == 3:         # mean-key landmark [n_phys][Hkv][128]: a stored bf16 code
        # Reading R24: the code is the exact mean rounded once to bf16 (the oracle's).  A kernel accumulating in fp32 may
        # land one bf16 step away, but only where the exact mean lies within the fp32 accumulation error of the rounding
        # boundary between the two codes -- the same kind of validity band R10 gives the top-k.  Anything else fails.
        ids = np.asarray(page_ids, np.int32)
        nv = None if n_valid is None else np.asarray(n_valid, np.int32)
        want = oracle.summarize_mean(h["k_cache"], ids, nv)
        got = _gpu_rows(summ_gpu, h, page_ids).contiguous().view(torch.int16).cpu().numpy().view(np.uint16)
        bad = np.nonzero(got != want)
        if len(bad[0]):
            exact, err = oracle.mean_landmark_band(h["k_cache"], ids, nv)
            g_, w_ = got[bad].astype(np.int64), want[bad].astype(np.int64)
            both_zero = ((g_ & 0x7FFF) == 0) & ((w_ & 0x7FFF) == 0)                          # +0 / -0
            assert (both_zero | (np.abs(g_ - w_) == 1)).all(), "mean landmark more than one bf16 step from the exact mean's code"
            val = lambda b: (b.astype(np.uint32) << 16).view(np.float32).astype(np.float64)
            mid = 0.5 * (val(got[bad]) + val(want[bad]))
            off = np.abs(exact[bad] - mid) - err[bad]
            assert (off[~both_zero] <= 0).all(), f"mean landmark differs outside the rounding band at {int((off > 0).sum())} entries"
        return dict(entries=int(got.size), one_step_apart=int(len(bad[0])))
    want = oracle.summarize(h["k_cache"], np.asarray(page_ids, np.int32), None if n_valid is None else np.asarray(n_valid, np.int32))
    got = bf16_to_f64(_gpu_rows(summ_gpu, h, page_ids))
    assert got.shape == want.shape
    bad = got != want
    assert not bad.any(), f"summaries differ at {int(bad.sum())} of {bad.size} entries"


def check_selection(res: dict, sel_gpu: np.ndarray, cnt_gpu: np.ndarray, seq_lens, scores_gpu=None, page_size: int = 16) -> dict:
    """res = oracle.sparse_step(...) for the same sequences.  Returns statistics."""
    n, Hkv, _ = sel_gpu.shape
    stats = dict(units=0, differing_units=0, band_pages=0)
    for i in range(n):
        L = int(seq_lens[i])
        n_pages = -(-L // page_size)
        cnt = int(res["sel_count"][i])
        assert int(cnt_gpu[i]) == cnt, f"seq {i}: sel_count {int(cnt_gpu[i])} != oracle {cnt}"
        F = set(np.flatnonzero(res["forced"][i, :n_pages]).tolist())
        for g in range(Hkv):
            got = sel_gpu[i, g, :cnt]
            want = res["sel"][i, g, :cnt]
            assert (np.diff(got) > 0).all(), f"seq {i} head {g}: list not strictly ascending"
            assert got[0] >= 0 and got[-1] < n_pages, f"seq {i} head {g}: page out of range"
            gs, ws = set(got.tolist()), set(want.tolist())
            assert F <= gs, f"seq {i} head {g}: forced pages missing: {sorted(F - gs)}"
            stats["units"] += 1
            diff = gs ^ ws
            if diff:
                stats["differing_units"] += 1
                tau = res["tau"][i, g]
                for p in diff:
                    s = res["scores"][i, g, p]
                    assert abs(s - tau) <= BAND_REL * abs(tau), (
                        f"seq {i} head {g}: page {p} differs outside the tie band: s={s!r} tau={tau!r}")
                    stats["band_pages"] += 1
            if scores_gpu is not None and not np.isnan(res["tau"][i, g]):
                cand = np.array(sorted(set(range(n_pages)) - F), dtype=np.int64)
                sg, so = scores_gpu[i, g, cand].astype(np.float64), res["scores"][i, g, cand]
                scale = np.abs(so).max() + 1e-30
                assert np.abs(sg - so).max() <= 2e-5 * scale, f"seq {i} head {g}: fp32 scores off by {np.abs(sg - so).max() / scale:.2e}"
    return stats


def check_outputs(out_gpu: torch.Tensor, lse_gpu, want_out: np.ndarray, want_lse: np.ndarray, what="out") -> dict:
    got = bf16_to_f64(out_gpu)
    err = np.abs(got - want_out)
    st = dict(max_abs=float(err.max()), mean_abs=float(err.mean()), rms_ref=float(np.sqrt((want_out ** 2).mean())))
    assert np.isfinite(got).all(), f"{what}: non-finite output"
    assert st["max_abs"] <= TOL_MAX_ABS and st["mean_abs"] <= TOL_MEAN_ABS, f"{what}: north_star tolerance exceeded {st}"
    over = err - (GATE_ABS + GATE_REL * np.abs(want_out))
    assert over.max() <= 0, f"{what}: internal elementwise gate exceeded by {over.max():.3e} {st}"
    assert st["mean_abs"] <= GATE_MEAN_ABS + 2.0 ** -9 * float(np.abs(want_out).mean()), f"{what}: internal mean gate exceeded {st}"
    if lse_gpu is not None:
        le = np.abs(lse_gpu.detach().cpu().numpy().astype(np.float64) - want_lse)
        st["lse_max_abs"] = float(le.max())
        assert st["lse_max_abs"] <= GATE_LSE_ABS, f"{what}: lse off by {st['lse_max_abs']:.3e}"
    return st


def check_sparse_step(eng, wl, h=None, idx=None, check_summ=True, out_idx=None) -> dict:
    """Full check of one engine step that has already run (summaries, sel_pages, sel_count, out, lse in `eng`).
    idx: optional subset of sequences to check (default: all).  out_idx: optional subset of idx whose out / lse are
    compared (default: all of idx); the selection, scores and summaries are checked on every sequence of idx."""
    h = h or wl.host()
    n = wl.n_seq
    idx = (np.asarray(h["seq_index"]) if "seq_index" in h else np.arange(n)) if idx is None else np.asarray(idx)
    hs = sub_host(h, idx)
    sched = oracle.Schedule.from_spec(eng.sched_spec)
    attend_all = out_idx is None
    if getattr(eng, "landmark", "minmax") == "mean":
        # O5..O8 on the stored landmark codes under test (verified against the exact mean's band by check_summaries)
        lm = (eng.summaries if hs["phys_ids"] is None else _gpu_rows(eng.summaries, hs, np.arange(len(hs["phys_ids"])))
              ).contiguous().view(torch.int16).cpu().numpy().view(np.uint16)
        res = oracle.sparse_step_mean(hs["q"], hs["k_cache"], hs["v_cache"], hs["page_table"], hs["seq_lens"], sched, wl.sm_scale,
                                      max_sel=eng.max_sel, landmarks=lm)
    else:
        res = oracle.sparse_step(hs["q"], hs["k_cache"], hs["v_cache"], hs["page_table"], hs["seq_lens"], sched, wl.sm_scale,
                                 max_sel=eng.max_sel, do_attention=attend_all)
    tidx = torch.as_tensor(idx).long().to(eng.out.device)
    sel_gpu = eng.sel_pages[tidx].cpu().numpy()
    cnt_gpu = eng.sel_count[tidx].cpu().numpy()
    scores_gpu = eng.scores[tidx].cpu().numpy() if eng.scores is not None else None
    P = getattr(wl, "page_size", 16)
    stats = check_selection(res, sel_gpu, cnt_gpu, hs["seq_lens"], scores_gpu, page_size=P)
    stats["seqs_selection"] = int(len(idx))
    if check_summ:
        # summaries of every page the checked sequences own (one sequence at a time: bounded host memory)
        for i in range(len(idx)):
            L = int(hs["seq_lens"][i]); npg = -(-L // P)
            v = np.full(npg, P, np.int32)
            if L % P: v[-1] = L % P
            check_summaries(eng.summaries, hs, hs["page_table"][i, :npg], v)
    if attend_all:
        pos = np.arange(len(idx))
    else:
        where = {int(s): j for j, s in enumerate(idx.tolist())}
        pos = np.array([where[int(s)] for s in out_idx], dtype=np.int64)
    stats["seqs_outputs"] = int(len(pos))
    if stats["differing_units"] or not attend_all:
        # R11: the oracle's attention evaluated on the GPU's own (validated) page sets -- identical to its own result
        # wherever the sets agree
        sel_fix = np.where(np.arange(sel_gpu.shape[2])[None, None, :] < cnt_gpu[:, None, None], sel_gpu, 0)[pos]
        want_out, want_lse = oracle.attention_on_sets(np.ascontiguousarray(hs["q"][pos]), hs["k_cache"], hs["v_cache"],
                                                      np.ascontiguousarray(hs["page_table"][pos]), np.ascontiguousarray(hs["seq_lens"][pos]),
                                                      np.ascontiguousarray(sel_fix), cnt_gpu[pos].astype(np.int64), wl.sm_scale)
    else:
        want_out, want_lse = res["out"], res["lse"]
    tpos = tidx[torch.as_tensor(pos).long().to(tidx.device)]
    stats.update(check_outputs(eng.out[tpos], eng.lse[tpos], want_out, want_lse, "sparse out"))
    return stats


def assert_same_result(out_a: torch.Tensor, out_b: torch.Tensor, what: str, lse_a=None, lse_b=None):
    """Two runs of the decode on the same inputs.  The kernel hands its tiles to whichever warp is free, so which tiles a
    warp sums is timing-dependent: the running maximum under which a probability is rounded to bf16 (2^-9 relative per term)
    and the fp32 summation order differ between two runs.  Both runs are valid evaluations, each within the arithmetic's own
    error of the exact result (the oracle gate: max-abs 3e-3), so they agree to about that error -- not bit for bit.
    Everything integer (page lists, counts) must be identical; the lse is summed in fp32 and agrees to fp32 rounding."""
    a, b = out_a.float(), out_b.float()
    tol = 2.0 ** -7 * torch.maximum(a.abs(), b.abs()) + 1.5e-3
    bad = (a - b).abs() > tol
    assert not bad.any(), f"{what}: {int(bad.sum())} outputs differ by more than the arithmetic's error between two runs"
    if lse_a is not None:
        assert (lse_a - lse_b).abs().max().item() <= 2e-5, f"{what}: lse differs between two runs"


def check_dense(eng, wl, h=None, idx=None) -> dict:
    h = h or wl.host()
    idx = (np.asarray(h["seq_index"]) if "seq_index" in h else np.arange(wl.n_seq)) if idx is None else np.asarray(idx)
    hs = sub_host(h, idx)
    want_out, want_lse = oracle.dense_step(hs["q"], hs["k_cache"], hs["v_cache"], hs["page_table"], hs["seq_lens"], wl.sm_scale)
    tidx = torch.as_tensor(idx).long().to(eng.out.device)
    return check_outputs(eng.out_dense[tidx], eng.lse_dense[tidx], want_out, want_lse, "dense out")
