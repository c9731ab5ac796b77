"""ctypes front end of ``sparrow_oracle.c`` (argument marshalling only; all arithmetic is in C).

TEST INFRASTRUCTURE: see the package docstring.  bf16 tensors are numpy ``uint16`` arrays of raw
bit patterns; everything the oracle returns is fp64 / integer numpy.
"""
from __future__ import annotations

import ctypes as C
import math
import os
import subprocess
from dataclasses import dataclass, field
from typing import Optional, Sequence

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "sparrow_oracle.c")
_LIB = os.path.join(_HERE, "libsparrow_oracle.so")
_lib = None

KIND = {"dense": 0, "fixed": 1, "clamp_frac": 2, "linear_frac": 3, "table": 4}


class _CSchedule(C.Structure):
    _fields_ = [
        ("kind", C.c_int32),
        ("sink_tokens", C.c_int32),
        ("local_tokens", C.c_int32),
        ("fixed_tokens", C.c_int64),
        ("floor_tokens", C.c_int64),
        ("f0_ppm", C.c_int64),
        ("f1_ppm", C.c_int64),
        ("L0", C.c_int64),
        ("L1", C.c_int64),
        ("table_pages", C.POINTER(C.c_int32)),
        ("table_len", C.c_int32),
        ("bin_tokens", C.c_int32),
    ]


@dataclass
class Schedule:
    """B(L) description, oracle side (R3).  Fractions are parts per million."""

    kind: str = "dense"
    sink_tokens: int = 0
    local_tokens: int = 0
    fixed_tokens: int = 0
    floor_tokens: int = 0
    f0_ppm: int = 0
    f1_ppm: int = 0
    L0: int = 0
    L1: int = 1
    table_pages: Sequence[int] = field(default_factory=tuple)
    bin_tokens: int = 2048

    @classmethod
    def from_spec(cls, spec: dict) -> "Schedule":
        """Build from the plain-data schedule dict of the workload generator."""
        return cls(**spec)

    def _c(self):
        tbl = np.ascontiguousarray(np.asarray(self.table_pages, dtype=np.int32))
        s = _CSchedule(
            KIND[self.kind], self.sink_tokens, self.local_tokens, self.fixed_tokens, self.floor_tokens,
            self.f0_ppm, self.f1_ppm, self.L0, self.L1,
            tbl.ctypes.data_as(C.POINTER(C.c_int32)), len(tbl), self.bin_tokens,
        )
        s._keep = tbl
        return s


def build(force: bool = False) -> str:
    """Compile the oracle with gcc (-O2, OpenMP).  Building the checker is not using it."""
    if force or not os.path.exists(_LIB) or os.path.getmtime(_LIB) < os.path.getmtime(_SRC):
        subprocess.check_call(
            ["gcc", "-O2", "-std=c11", "-fopenmp", "-fPIC", "-shared", "-o", _LIB, _SRC, "-lm"]
        )
    return _LIB


def _load():
    global _lib
    if _lib is None:
        build()
        _lib = C.CDLL(_LIB)
        _lib.oracle_budget_tokens.restype = C.c_int64
        _lib.oracle_k_pages.restype = C.c_int64
        _lib.oracle_forced_pages.restype = C.c_int64
        _lib.oracle_select_unit.restype = C.c_int64
        _lib.oracle_sparse_step.restype = C.c_int
        _lib.oracle_num_threads.restype = C.c_int
    return _lib


def _p(a: Optional[np.ndarray]):
    return None if a is None else a.ctypes.data_as(C.c_void_p)


def _u16(a) -> np.ndarray:
    a = np.ascontiguousarray(a)
    assert a.dtype == np.uint16, "bf16 tensors are passed as uint16 bit patterns"
    return a


def _i32(a) -> np.ndarray:
    return np.ascontiguousarray(np.asarray(a, dtype=np.int32))


def _i64(x):
    return C.c_int64(int(x))


def num_threads() -> int:
    return int(_load().oracle_num_threads())


def budget_tokens(sched: Schedule, L: int, page_size: int = 16) -> int:
    s = sched._c()
    return int(_load().oracle_budget_tokens(C.byref(s), _i64(L), _i64(page_size)))


def k_pages(sched: Schedule, L: int, page_size: int = 16) -> int:
    s = sched._c()
    return int(_load().oracle_k_pages(C.byref(s), _i64(L), _i64(page_size)))


def forced_pages(L: int, S: int, W: int, page_size: int = 16) -> np.ndarray:
    n_pages = -(-L // page_size)
    f = np.zeros(max(n_pages, 1), dtype=np.uint8)
    _load().oracle_forced_pages(_i64(L), _i64(S), _i64(W), _i64(page_size), _p(f))
    return f[:n_pages].astype(bool)


def summarize(k_cache, page_ids, n_valid=None) -> np.ndarray:
    """O1.  k_cache [n_phys][Hkv][P][D] uint16 -> [n_update][Hkv][2][D] float64 (min, max)."""
    k_cache = _u16(k_cache)
    _, Hkv, P, D = k_cache.shape
    page_ids = _i32(page_ids)
    nv = None if n_valid is None else _i32(n_valid)
    out = np.empty((len(page_ids), Hkv, 2, D), dtype=np.float64)
    _load().oracle_summarize(_p(k_cache), _p(page_ids), _p(nv), _i64(len(page_ids)), _i64(Hkv), _i64(P), _i64(D), _p(out))
    return out


def scores_unit(q_seq, k_cache, pt_row, L: int, g: int) -> np.ndarray:
    """O5 for one (sequence, kv-head): scores of all n_pages(L) logical pages."""
    q_seq, k_cache, pt_row = _u16(q_seq), _u16(k_cache), _i32(pt_row)
    Hq, D = q_seq.shape
    _, Hkv, P, _ = k_cache.shape
    n_pages = -(-L // P)
    s = np.empty(n_pages, dtype=np.float64)
    _load().oracle_scores_unit(_p(q_seq), _p(k_cache), _p(pt_row), _i64(L), _i64(g), _i64(Hq), _i64(Hkv), _i64(P), _i64(D), _p(s))
    return s


def select_unit(scores, forced, K_pages: int):
    """O4, O6, O7 for one (sequence, kv-head).  Returns (ascending page list, tau)."""
    scores = np.ascontiguousarray(scores, dtype=np.float64)
    forced = np.ascontiguousarray(np.asarray(forced, dtype=np.uint8))
    n_pages = len(forced)
    sel = np.empty(max(n_pages, 1), dtype=np.int32)
    tau = C.c_double()
    m = _load().oracle_select_unit(_p(scores), _p(forced), _i64(n_pages), _i64(K_pages), _p(sel), C.byref(tau))
    return sel[:m].copy(), float(tau.value)


def attention_unit(q_seq, k_cache, v_cache, pt_row, L: int, pages, g: int, sm_scale: float, want_probs: bool = False):
    """O8 for one (sequence, kv-head).  Returns (out [r][D], lse [r][, probs [r][n_sel*P]])."""
    q_seq, k_cache, v_cache, pt_row, pages = _u16(q_seq), _u16(k_cache), _u16(v_cache), _i32(pt_row), _i32(pages)
    Hq, D = q_seq.shape
    _, Hkv, P, _ = k_cache.shape
    r = Hq // Hkv
    out = np.empty((r, D), dtype=np.float64)
    lse = np.empty(r, dtype=np.float64)
    probs = np.zeros((r, max(len(pages) * P, 1)), dtype=np.float64) if want_probs else None
    _load().oracle_attention_unit(
        _p(q_seq), _p(k_cache), _p(v_cache), _p(pt_row), _i64(L), _p(pages), _i64(len(pages)), _i64(g),
        _i64(Hq), _i64(Hkv), _i64(P), _i64(D), C.c_double(sm_scale), _p(out), _p(lse), _p(probs))
    if want_probs:
        return out, lse, probs[:, : len(pages) * P]
    return out, lse


def attention_partial_unit(q_seq, k_cache, v_cache, pt_row, L: int, pages, g: int, sm_scale: float):
    """a6 partial state (m [r], l [r], o [r][D]) of one chunk of pages."""
    q_seq, k_cache, v_cache, pt_row, pages = _u16(q_seq), _u16(k_cache), _u16(v_cache), _i32(pt_row), _i32(pages)
    Hq, D = q_seq.shape
    _, Hkv, P, _ = k_cache.shape
    r = Hq // Hkv
    m = np.empty(r, dtype=np.float64)
    l = np.empty(r, dtype=np.float64)
    o = np.empty((r, D), dtype=np.float64)
    _load().oracle_attention_partial_unit(
        _p(q_seq), _p(k_cache), _p(v_cache), _p(pt_row), _i64(L), _p(pages), _i64(len(pages)), _i64(g),
        _i64(Hq), _i64(Hkv), _i64(P), _i64(D), C.c_double(sm_scale), _p(m), _p(l), _p(o))
    return m, l, o


def lse_merge(m_i, l_i, o_i):
    """a7 for one query head: partials m_i [n], l_i [n], o_i [n][D] -> (out [D], lse)."""
    m_i = np.ascontiguousarray(m_i, dtype=np.float64)
    l_i = np.ascontiguousarray(l_i, dtype=np.float64)
    o_i = np.ascontiguousarray(o_i, dtype=np.float64)
    n, D = o_i.shape
    out = np.empty(D, dtype=np.float64)
    lse = C.c_double()
    _load().oracle_lse_merge(_p(m_i), _p(l_i), _p(o_i), _i64(n), _i64(D), _p(out), C.byref(lse))
    return out, float(lse.value)


def sparse_step(q, k_cache, v_cache, page_table, seq_lens, sched: Schedule, sm_scale: float,
                max_sel: Optional[int] = None, do_attention: bool = True) -> dict:
    """O1..O8 for a batch.  Returns a dict with every intermediate the checker needs."""
    q, k_cache, v_cache = _u16(q), _u16(k_cache), _u16(v_cache)
    page_table, seq_lens = _i32(page_table), _i32(seq_lens)
    n, Hq, D = q.shape
    _, Hkv, P, _ = k_cache.shape
    max_pages = page_table.shape[1]
    if max_sel is None:
        max_sel = max_pages
    res = dict(
        budget_tokens=np.zeros(n, dtype=np.int64),
        k_pages=np.zeros(n, dtype=np.int64),
        sel_count=np.zeros(n, dtype=np.int64),
        forced=np.zeros((n, max_pages), dtype=np.uint8),
        scores=np.zeros((n, Hkv, max_pages), dtype=np.float64),
        tau=np.zeros((n, Hkv), dtype=np.float64),
        sel=np.zeros((n, Hkv, max_sel), dtype=np.int32),
        out=np.zeros((n, Hq, D), dtype=np.float64),
        lse=np.zeros((n, Hq), dtype=np.float64),
    )
    s = sched._c()
    rc = _load().oracle_sparse_step(
        _p(q), _p(k_cache), _p(v_cache), _p(page_table), _p(seq_lens), C.byref(s),
        _i64(n), _i64(Hq), _i64(Hkv), _i64(P), _i64(D), _i64(max_pages), _i64(max_sel),
        C.c_double(sm_scale), C.c_int(1 if do_attention else 0),
        _p(res["budget_tokens"]), _p(res["k_pages"]), _p(res["sel_count"]), _p(res["forced"]),
        _p(res["scores"]), _p(res["tau"]), _p(res["sel"]), _p(res["out"]), _p(res["lse"]))
    if rc != 0:
        raise ValueError("oracle_sparse_step: max_sel too small for the schedule")
    return res


def attention_on_sets(q, k_cache, v_cache, page_table, seq_lens, sel, sel_count, sm_scale: float):
    """O8 on caller-supplied page lists sel [n][Hkv][max_sel] (R11).  Returns (out, lse)."""
    q, k_cache, v_cache = _u16(q), _u16(k_cache), _u16(v_cache)
    page_table, seq_lens, sel = _i32(page_table), _i32(seq_lens), _i32(sel)
    sel_count = np.ascontiguousarray(np.asarray(sel_count, dtype=np.int64))
    n, Hq, D = q.shape
    _, Hkv, P, _ = k_cache.shape
    out = np.zeros((n, Hq, D), dtype=np.float64)
    lse = np.zeros((n, Hq), dtype=np.float64)
    _load().oracle_attention_on_sets(
        _p(q), _p(k_cache), _p(v_cache), _p(page_table), _p(seq_lens), _p(sel), _p(sel_count),
        _i64(n), _i64(Hq), _i64(Hkv), _i64(P), _i64(D), _i64(page_table.shape[1]), _i64(sel.shape[2]),
        C.c_double(sm_scale), _p(out), _p(lse))
    return out, lse


def dense_step(q, k_cache, v_cache, page_table, seq_lens, sm_scale: float):
    """a8: dense attention over all pages.  Returns (out [n][Hq][D], lse [n][Hq])."""
    q, k_cache, v_cache = _u16(q), _u16(k_cache), _u16(v_cache)
    page_table, seq_lens = _i32(page_table), _i32(seq_lens)
    n, Hq, D = q.shape
    _, Hkv, P, _ = k_cache.shape
    out = np.zeros((n, Hq, D), dtype=np.float64)
    lse = np.zeros((n, Hq), dtype=np.float64)
    _load().oracle_dense_step(
        _p(q), _p(k_cache), _p(v_cache), _p(page_table), _p(seq_lens),
        _i64(n), _i64(Hq), _i64(Hkv), _i64(P), _i64(D), _i64(page_table.shape[1]), C.c_double(sm_scale),
        _p(out), _p(lse))
    return out, lse


# ---------------------------------------------------------------------------------------------------------------
# the multi-step rollout loop.  PAPER.md:138-147 -- every generated token runs landmark scoring ->
# Top-k -> attention over the budget; PAPER.md:109-119 -- the budget follows the growing sequence length; the cache
# side (the token's K/V appended at position L, landmarks of pages that fill) is what any paged decode does.  Written
# out step by step with the functions above; plain numpy indexing for the data movement.
def append_step(k_cache, v_cache, page_table, seq_lens, k_new, v_new, page_size: int = 16):
    """In place: token i's K/V rows go to position L_i (logical page L_i // 16 through the page table, row L_i % 16),
    then L_i += 1.  Returns the physical pages that became full (their landmarks are due, a1 'on page fill')."""
    filled = []
    for i in range(len(seq_lens)):
        L = int(seq_lens[i])
        page = int(page_table[i, L // page_size])
        k_cache[page, :, L % page_size, :] = k_new[i]
        v_cache[page, :, L % page_size, :] = v_new[i]
        seq_lens[i] = L + 1
        if (L + 1) % page_size == 0:
            filled.append(page)
    return filled


def rollout(q_steps, k_steps, v_steps, k_cache, v_cache, page_table, seq_lens, sched: Optional[Schedule], sm_scale: float,
            max_sel: Optional[int] = None):
    """T decode steps: append the step's K/V, then O1..O8 (sched given) or dense attention (sched None) with the
    step's query over the grown cache.  Inputs are not modified.  Returns one dict per step: sparse_step's result
    (or {'out', 'lse'} for dense) plus 'seq_lens' and 'filled' (physical pages whose landmarks were (re)built)."""
    q_steps, k_steps, v_steps = _u16(q_steps), _u16(k_steps), _u16(v_steps)
    k_cache, v_cache = _u16(k_cache).copy(), _u16(v_cache).copy()
    page_table, seq_lens = _i32(page_table), _i32(seq_lens).copy()
    steps = []
    for t in range(q_steps.shape[0]):
        filled = append_step(k_cache, v_cache, page_table, seq_lens, k_steps[t], v_steps[t], page_size=k_cache.shape[2])
        if sched is None:
            out, lse = dense_step(q_steps[t], k_cache, v_cache, page_table, seq_lens, sm_scale)
            res = dict(out=out, lse=lse)
        else:
            res = sparse_step(q_steps[t], k_cache, v_cache, page_table, seq_lens, sched, sm_scale, max_sel=max_sel)
        res["seq_lens"] = seq_lens.copy()
        res["filled"] = filled
        steps.append(res)
    return steps, k_cache, v_cache


# ---------------------------------------------------------------------------------------------------------------
# the paper's rollout cost model, restated from PAPER.md:129-145 (Eq. 2-3) and :474-498 (App. F)
# in the paper's notation.  Plain Python floats (fp64).
def cost_model(P, B, N, L_in, L_out, D, r, I, K, pagesize, c=1.0) -> dict:
    """P parameters, B batch, N samples, L_in prompt, L_out response, D K/V width, r GQA ratio, I hardware intensity
    (R18), K KV budget in tokens, c landmark vectors per page (1 in the paper's model; R1 uses 2).
    App. F:  L_dense = min(L_out, K - L_in) (not below 0);  H = (2 L_in + L_dense) L_dense + 2 K (L_out - L_dense)+
             C_comp = 2 P B N L_out + r B N (2 L_in + L_out) L_out D;  C_mem = 2 P L_out + B N (2 L_in L_out + L_out^2) D
             sparse: the attention terms with H in place of (2 L_in + L_out) L_out.
    Eq. 3 scoring (reading R21: one landmark visit per page of the context per decode step, only on the steps decoded
    under the budget): visits S = sum over those steps of (L_in + t) / pagesize (continuous form, as the paper's
    L_out^2 / 2 terms).  The paper charges one D-vector read (memory D) and r D multiply-adds (compute r D) per landmark
    vector visited -- its clean terms at :142 are memory I N D L_out^2 / (2 pagesize), compute r N D L_out^2 / (2 pagesize),
    the same r : 1 ratio as the attention terms -- so with c landmark vectors per page:
    memory c B N D S;  compute r c B N D S.   C = C_comp + I C_mem.
    "parity unpinned": the L_in part of S.  PAPER.md:142 prints its L_in scoring terms without the 1 / pagesize factor; R21
    reads that as garbled, and the only pin of these terms is a per-step sum written from the same reading."""
    L_dense = min(L_out, max(K - L_in, 0.0))
    H = (2 * L_in + L_dense) * L_dense + 2 * K * max(L_out - L_dense, 0.0)
    H_dense = (2 * L_in + L_out) * L_out
    S = ((L_in * L_out + L_out ** 2 / 2) - (L_in * L_dense + L_dense ** 2 / 2)) / pagesize
    dense_comp = 2 * P * B * N * L_out + r * B * N * H_dense * D
    dense_mem = 2 * P * L_out + B * N * H_dense * D
    sparse_comp = 2 * P * B * N * L_out + r * B * N * D * H
    sparse_mem = 2 * P * L_out + B * N * D * H
    scoring_comp = r * c * B * N * D * S
    scoring_mem = c * B * N * D * S
    return dict(attn_elems_dense=H_dense, attn_elems_sparse=H, landmark_visits=S, dense_comp=dense_comp, dense_mem=dense_mem,
                dense_total=dense_comp + I * dense_mem, sparse_comp=sparse_comp, sparse_mem=sparse_mem,
                scoring_comp=scoring_comp, scoring_mem=scoring_mem,
                sparse_total=sparse_comp + scoring_comp + I * (sparse_mem + scoring_mem))


# ---------------------------------------------------------------------------------------------------------------
# the paper's divergence statistic.  PAPER.md:76-79 (Eq. 1): alpha = E_{x~Q}[min(p(x)/q(x), 1)]
# = sum_x min(p(x), q(x)); approximated from the top-20 tokens and logprobs per position; PAPER.md:101,
# :119: tokens grouped by position in 2K bins, the statistic is the 5-percentile per bin.  fp64, plain loops.
def acceptance_rate(ids_p, logp_p, ids_q, logp_q) -> np.ndarray:
    """alpha per position from the two top-N lists ([n_pos][N] token ids and natural-log probabilities): the sum of
    min(p, q) over the tokens present in both lists (reading R23: a token missing from a list adds nothing)."""
    ids_p, ids_q = np.asarray(ids_p), np.asarray(ids_q)
    p, q = np.exp(np.asarray(logp_p, dtype=np.float64)), np.exp(np.asarray(logp_q, dtype=np.float64))
    alpha = np.zeros(len(ids_p), dtype=np.float64)
    for i in range(len(ids_p)):
        where_q = {int(t): j for j, t in enumerate(ids_q[i])}
        for j, t in enumerate(ids_p[i]):
            k = where_q.get(int(t))
            if k is not None:
                alpha[i] += min(p[i, j], q[i, k])
    return alpha


def binned_quantile(alpha, positions, bin_tokens: int, n_bins: int, quantile: float):
    """Per length bin b = min(position // bin_tokens, n_bins - 1): (count, nearest-rank quantile) = the value of rank
    max(1, ceil(quantile * count)) of the bin's alphas in ascending order; NaN for an empty bin."""
    alpha, positions = np.asarray(alpha, dtype=np.float64), np.asarray(positions)
    b = np.minimum(np.maximum(positions // bin_tokens, 0), n_bins - 1)
    counts = np.zeros(n_bins, dtype=np.int64)
    out = np.full(n_bins, np.nan)
    for k in range(n_bins):
        v = np.sort(alpha[b == k])
        counts[k] = len(v)
        if len(v):
            out[k] = v[max(1, math.ceil(quantile * len(v))) - 1]
    return counts, out


# ---------------------------------------------------------------------------------------------------------------
# SURVEY.md 8(f)-2, landmark variant: ONE vector per page, the mean key -- the landmark the paper's cost model charges
# (D elements per page; the form itself is left open at :147, reading R1).  Plain definition (reading
# R24): the arithmetic mean of the page's valid keys, evaluated in fp64 (a sum of at most 128 bf16 values is exact in
# fp64 unless their exponents span more than 40 binades) and rounded ONCE to bf16, nearest even.  Everything after it
# (score, top-k, attention) is fp64 as in O5..O8.
def _round_to_bf16_bits(x: np.ndarray) -> np.ndarray:
    """fp64 -> nearest bf16 (8 significant bits, ties to even), returned as the bf16 BIT pattern.  Written on the
    significand directly so that there is one rounding only (fp64 -> fp32 -> bf16 would round twice)."""
    x = np.asarray(x, dtype=np.float64)
    m, e = np.frexp(x)                                   # x = m * 2^e, 0.5 <= |m| < 1
    y = np.ldexp(np.rint(np.ldexp(m, 8)), e - 8)         # rint rounds halves to even; 8 bits of significand kept
    assert (np.abs(y[y != 0]) >= 2.0 ** -126).all(), "bf16 subnormals are outside this oracle's scope"
    return (y.astype(np.float32).view(np.uint32) >> 16).astype(np.uint16)      # y is exactly representable: no rounding here


def summarize_mean(k_cache, page_ids, n_valid=None) -> np.ndarray:
    """k_cache [n_phys][Hkv][P][D] uint16 (bf16 bits) -> mean-key landmarks [n_update][Hkv][D] as bf16 BITS (uint16):
    mean over the page's valid tokens (fp64), rounded once to bf16."""
    k_cache = _u16(k_cache)
    P = k_cache.shape[2]
    out = np.zeros((len(page_ids), k_cache.shape[1], k_cache.shape[3]), dtype=np.uint16)
    for u, page in enumerate(page_ids):
        valid = P if n_valid is None else int(n_valid[u])
        rows = (k_cache[int(page)].astype(np.uint32) << 16).view(np.float32).astype(np.float64)   # [Hkv][P][D]
        acc = np.zeros((rows.shape[0], rows.shape[2]), dtype=np.float64)
        for t in range(valid):
            acc = acc + rows[:, t, :]
        out[u] = _round_to_bf16_bits(acc / float(max(valid, 1)))
    return out


def mean_landmark_band(k_cache, page_ids, n_valid=None):
    """For a checker: (exact fp64 mean, fp32-accumulation error bound) per landmark entry, [n_update][Hkv][D] each.
    A kernel that accumulates the page's keys in fp32 (any order) and divides in fp32 returns a value within
    err = (valid + 1) * 2^-24 * mean_t |k_t| of the exact mean, so its bf16 code may differ from summarize_mean's by
    one step only where the exact mean lies within err of the rounding boundary between the two codes (reading R24)."""
    k_cache = _u16(k_cache)
    P = k_cache.shape[2]
    shape = (len(page_ids), k_cache.shape[1], k_cache.shape[3])
    exact, err = np.zeros(shape), np.zeros(shape)
    for u, page in enumerate(page_ids):
        valid = P if n_valid is None else int(n_valid[u])
        rows = (k_cache[int(page)].astype(np.uint32) << 16).view(np.float32).astype(np.float64)[:, :valid, :]
        exact[u] = rows.sum(1) / float(max(valid, 1))
        err[u] = (valid + 1) * 2.0 ** -24 * np.abs(rows).sum(1) / float(max(valid, 1))
    return exact, err


def sparse_step_mean(q, k_cache, v_cache, page_table, seq_lens, sched: Schedule, sm_scale: float, max_sel: Optional[int] = None,
                     landmarks=None) -> dict:
    """O1..O8 with the mean-key landmark: score s[p] = sum_{h in group} q_h . mean[p] (fp64 over the bf16 landmark);
    budget, forced pages, top-k (ties to the lower page) and attention exactly as sparse_step.
    landmarks: optional stored codes [n_phys][Hkv][D] (bf16 bits) to score with instead of summarize_mean's -- a
    checker passes the codes under test once it has verified them against mean_landmark_band, so that O5..O8 are
    compared on the same stored landmarks (as R11 does for the attention on the selected sets)."""
    q, k_cache, v_cache = _u16(q), _u16(k_cache), _u16(v_cache)
    page_table, seq_lens = _i32(page_table), _i32(seq_lens)
    n, Hq, D = q.shape
    _, Hkv, P, _ = k_cache.shape
    r = Hq // Hkv
    max_pages = page_table.shape[1]
    max_sel = max_pages if max_sel is None else max_sel
    qf = (q.astype(np.uint32) << 16).view(np.float32).astype(np.float64)
    res = dict(k_pages=np.zeros(n, np.int64), sel_count=np.zeros(n, np.int64), forced=np.zeros((n, max_pages), np.uint8),
               scores=np.zeros((n, Hkv, max_pages)), tau=np.full((n, Hkv), np.nan), sel=np.zeros((n, Hkv, max_sel), np.int32))
    for i in range(n):
        L = int(seq_lens[i]); n_pages = -(-L // P)
        K = k_pages(sched, L, P)
        F = forced_pages(L, sched.sink_tokens, sched.local_tokens, P)
        res["k_pages"][i] = K
        res["forced"][i, :n_pages] = F
        nv = np.full(n_pages, P, np.int32)
        if L % P:
            nv[-1] = L % P
        lm_bits = summarize_mean(k_cache, page_table[i, :n_pages], nv) if landmarks is None else _u16(landmarks)[page_table[i, :n_pages]]
        lm = (lm_bits.astype(np.uint32) << 16).view(np.float32).astype(np.float64)
        for g in range(Hkv):
            s = lm[:, g, :] @ qf[i, g * r:(g + 1) * r].sum(0)
            res["scores"][i, g, :n_pages] = s
            if K >= n_pages:
                sel = np.arange(n_pages)
            else:
                cand = np.flatnonzero(F == 0)
                k = max(0, K - int(F.sum()))
                order = sorted(cand.tolist(), key=lambda p: (-s[p], p))[:k]
                if k > 0:
                    res["tau"][i, g] = s[order[-1]]
                sel = np.sort(np.concatenate([np.flatnonzero(F), np.array(order, dtype=np.int64)]))
            res["sel_count"][i] = len(sel)
            res["sel"][i, g, :len(sel)] = sel
    res["out"], res["lse"] = attention_on_sets(q, k_cache, v_cache, page_table, seq_lens, res["sel"], res["sel_count"], sm_scale)
    return res
