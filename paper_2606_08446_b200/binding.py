"""Thin ctypes binding of libsparrow_b200.so: same names as include/sparrow.h, argument marshalling only.

Every step of the path runs in the CUDA kernels.  torch is used for device memory and streams.  There is no
CPU fallback: if the shared library is missing this module raises at import, and a non-zero status raises
``SparrowError``.
"""
from __future__ import annotations

import ctypes as C
import os
from typing import Optional

import torch

_HERE = os.path.dirname(os.path.abspath(__file__))
# SPARROW_B200_LIB names another build of this same library (the tracing build, libsparrow_b200_trace.so: build.py --trace)
LIB_PATH = os.environ.get("SPARROW_B200_LIB") or os.path.join(_HERE, "libsparrow_b200.so")
if not os.path.exists(LIB_PATH):
    raise ImportError(
        f"{LIB_PATH} is missing: build it with `python -m paper_2606_08446_b200.build` "
        "(or __graft_entry__.build()); there is no fallback path")
_lib = C.CDLL(LIB_PATH)

SCHED_KIND = {"dense": 0, "fixed": 1, "clamp_frac": 2, "linear_frac": 3, "table": 4}


class SparrowError(RuntimeError):
    pass


class sparrow_shape_t(C.Structure):
    _fields_ = [("n_seq", C.c_int32), ("n_q_heads", C.c_int32), ("n_kv_heads", C.c_int32), ("head_dim", C.c_int32),
                ("page_size", C.c_int32), ("max_pages_per_seq", C.c_int32), ("n_phys_pages", C.c_int64), ("landmark", C.c_int32),
                ("flags", C.c_int32), ("kv_stride_page", C.c_int64), ("kv_stride_head", C.c_int64), ("kv_stride_tok", C.c_int64)]


class sparrow_schedule_t(C.Structure):
    _fields_ = [("kind", C.c_int32), ("sink_tokens", C.c_int32), ("local_tokens", C.c_int32),
                ("fixed_tokens", C.c_int64), ("floor_tokens", C.c_int64), ("f0_ppm", C.c_int64), ("f1_ppm", C.c_int64),
                ("L0", C.c_int64), ("L1", C.c_int64), ("table_pages", C.POINTER(C.c_int32)),
                ("table_len", C.c_int32), ("bin_tokens", C.c_int32), ("page_size", C.c_int32)]


class sparrow_cost_args_t(C.Structure):
    _fields_ = [(k, C.c_double) for k in ("params", "batch_size", "n_samples", "L_in", "L_out", "D", "r", "intensity",
                                          "budget_tokens", "page_size", "landmarks_per_page")]


class sparrow_cost_t(C.Structure):
    _fields_ = [(k, C.c_double) for k in ("attn_elems_dense", "attn_elems_sparse", "landmark_visits", "dense_comp", "dense_mem",
                                          "dense_total", "sparse_comp", "sparse_mem", "scoring_comp", "scoring_mem", "sparse_total")]


LANDMARK = {"minmax": 0, "mean": 1}


FLAG_DETERMINISTIC = 1


def make_shape(n_seq, n_q_heads, n_kv_heads, max_pages_per_seq, n_phys_pages, head_dim=128, page_size=16, landmark="minmax",
               kv_layout="hnd", deterministic=False):
    """kv_layout: "hnd" (packed [page][kv-head][token][128], strides left 0), "nhd" ([page][token][kv-head][128]) or a tuple
    (stride_page, stride_head, stride_tok) in elements."""
    if kv_layout == "hnd":
        st = (0, 0, 0)
    elif kv_layout == "nhd":
        st = (page_size * n_kv_heads * head_dim, head_dim, n_kv_heads * head_dim)
    else:
        st = tuple(int(x) for x in kv_layout)
    return sparrow_shape_t(n_seq, n_q_heads, n_kv_heads, head_dim, page_size, max_pages_per_seq, n_phys_pages, LANDMARK[landmark],
                           FLAG_DETERMINISTIC if deterministic else 0, *st)


def make_schedule(spec: dict, page_size: int = 0) -> sparrow_schedule_t:
    """From the plain-data schedule dict of ``workloads`` (kind, sink_tokens, ... table_pages, bin_tokens)."""
    tbl = (C.c_int32 * max(1, len(spec.get("table_pages", ()))))(*spec.get("table_pages", ()))
    s = sparrow_schedule_t(SCHED_KIND[spec["kind"]], spec.get("sink_tokens", 0), spec.get("local_tokens", 0),
                           spec.get("fixed_tokens", 0), spec.get("floor_tokens", 0), spec.get("f0_ppm", 0),
                           spec.get("f1_ppm", 0), spec.get("L0", 0), spec.get("L1", 1),
                           C.cast(tbl, C.POINTER(C.c_int32)), len(spec.get("table_pages", ())), spec.get("bin_tokens", 2048),
                           spec.get("page_size", page_size))
    s._keep = tbl
    return s


_vp, _i32, _i64, _sz, _f = C.c_void_p, C.c_int32, C.c_int64, C.c_size_t, C.c_float
_SHP, _SCH = C.POINTER(sparrow_shape_t), C.POINTER(sparrow_schedule_t)
_SIGS = {
    "sparrow_summarize": (C.c_int, [_vp, _vp, _vp, _vp, _i64, _SHP, _vp]),
    "sparrow_select": (C.c_int, [_vp, _vp, _vp, _vp, _SCH, _vp, _i32, _vp, _vp, _vp, _sz, _SHP, _vp]),
    "sparrow_select_static": (C.c_int, [_vp, _vp, _vp, _vp, _SCH, _vp, _i32, _vp, _vp, _SHP, _vp]),
    "sparrow_select_static_bytes": (_sz, []),
    "sparrow_sparse_decode": (C.c_int, [_vp, _vp, _vp, _vp, _vp, _vp, _i32, _vp, _vp, _vp, _f, _vp, _sz, _SHP, _vp]),
    "sparrow_dense_decode": (C.c_int, [_vp, _vp, _vp, _vp, _vp, _vp, _vp, _f, _vp, _sz, _SHP, _vp]),
    "sparrow_append": (C.c_int, [_vp, _vp, _vp, _vp, _vp, _vp, _vp, _SHP, _vp]),
    "sparrow_step_host": (C.c_int, [_vp, _i64, C.c_int, _vp, _vp, _vp, _vp, _SCH, _i32, _f, _vp, _vp, _sz, _SHP, _vp]),
    "sparrow_step_host_async": (C.c_int, [_vp, _i64, C.c_int, _vp, _vp, _vp, _vp, _SCH, _i32, _f, _vp, _vp, _sz, _SHP, _vp]),
    "sparrow_step_host_block_bytes": (_sz, [_SHP, C.POINTER(_sz), C.POINTER(_sz), C.POINTER(_sz)]),
    "sparrow_select_workspace_bytes": (_sz, [_SHP]),
    "sparrow_decode_workspace_bytes": (_sz, [_SHP, _i32]),
    "sparrow_step_scratch_bytes": (_sz, [_SHP, _i32]),
    "sparrow_acceptance": (C.c_int, [_vp, _vp, _vp, _vp, _vp, _i64, _i32, _i32, _i32, _f, _vp, _vp, _vp, _vp, _sz, _vp]),
    "sparrow_acceptance_workspace_bytes": (_sz, [_i32]),
    "sparrow_cost_model": (C.c_int, [C.POINTER(sparrow_cost_args_t), C.POINTER(sparrow_cost_t)]),
    "sparrow_budget_tokens": (_i64, [_SCH, _i64]),
    "sparrow_k_pages": (_i32, [_SCH, _i64]),
    "sparrow_forced_count": (_i32, [_SCH, _i64]),
    "sparrow_sel_count": (_i32, [_SCH, _i64]),
    "sparrow_max_sel_pages": (_i32, [_SCH, _i64]),
    "sparrow_strerror": (C.c_char_p, [C.c_int]),
    "sparrow_version": (C.c_int, []),
    "sparrow_last_launch_count": (C.c_int, []),
    "sparrow_trace_set": (C.c_int, [_vp]),
}
for _name, (_res, _args) in _SIGS.items():
    _fn = getattr(_lib, _name)          # AttributeError here = the library does not export a declared symbol
    _fn.restype, _fn.argtypes = _res, _args
EXPORTS = tuple(_SIGS)
# the struct layouts above are those of ABI 300 (include/sparrow.h: SPARROW_ABI_VERSION); a library built from another header
# would read garbage strides out of a shorter or longer sparrow_shape_t
ABI_VERSION = 300
if _lib.sparrow_version() != ABI_VERSION:
    raise ImportError(f"{LIB_PATH} reports ABI {_lib.sparrow_version()}, this binding is written for {ABI_VERSION}: rebuild it "
                      "(`python -m paper_2606_08446_b200.build --force`)")


def _check(rc: int, what: str):
    if rc != 0:
        raise SparrowError(f"{what}: {_lib.sparrow_strerror(rc).decode()} (status {rc})")


def _ptr(t: Optional[torch.Tensor], *, cuda: bool = True):
    if t is None:
        return None
    assert t.is_contiguous(), "tensors must be contiguous"
    if cuda:
        assert t.is_cuda, "device pointer expected"
    return C.c_void_p(t.data_ptr())


def _stream(stream):
    if stream is None:
        stream = torch.cuda.current_stream()
    return C.c_void_p(stream.cuda_stream)


def _by(x):
    return C.byref(x)


def sparrow_version() -> int:
    return _lib.sparrow_version()


def sparrow_trace_set(buffer: Optional[torch.Tensor]):
    """Tracing build only: point the kernels' stamps at `buffer` (int64 [65536][8] on the device, zeroed) or switch them off."""
    if buffer is not None:
        assert buffer.is_cuda and buffer.dtype == torch.int64 and buffer.numel() >= 65536 * 8 and buffer.is_contiguous()
    _check(_lib.sparrow_trace_set(_ptr(buffer)), "sparrow_trace_set")


def sparrow_last_launch_count() -> int:
    return _lib.sparrow_last_launch_count()


def sparrow_strerror(rc: int) -> str:
    return _lib.sparrow_strerror(rc).decode()


def sparrow_select_workspace_bytes(shape) -> int:
    return _lib.sparrow_select_workspace_bytes(_by(shape))


def sparrow_decode_workspace_bytes(shape, max_sel: int) -> int:
    return _lib.sparrow_decode_workspace_bytes(_by(shape), max_sel)


def sparrow_step_scratch_bytes(shape, max_sel: int) -> int:
    return _lib.sparrow_step_scratch_bytes(_by(shape), max_sel)


def sparrow_acceptance_workspace_bytes(n_bins: int) -> int:
    return _lib.sparrow_acceptance_workspace_bytes(n_bins)


def sparrow_acceptance(ids_p, logp_p, ids_q, logp_q, positions, top_n: int, bin_tokens: int, n_bins: int, quantile: float,
                       alpha, bin_quantile, bin_count, workspace, stream=None, *, check=True):
    rc = _lib.sparrow_acceptance(_ptr(ids_p), _ptr(logp_p), _ptr(ids_q), _ptr(logp_q), _ptr(positions), int(positions.numel()),
                                 top_n, bin_tokens, n_bins, quantile, _ptr(alpha), _ptr(bin_quantile), _ptr(bin_count),
                                 _ptr(workspace), 0 if workspace is None else workspace.numel() * workspace.element_size(),
                                 _stream(stream))
    if check:
        _check(rc, "sparrow_acceptance")
    return rc


def sparrow_cost_model(*, check=True, **kw) -> dict:
    """Eq. 2-3 / App. F of the paper; keyword arguments = the fields of sparrow_cost_args_t.  Returns a dict."""
    args, cost = sparrow_cost_args_t(**{k: float(v) for k, v in kw.items()}), sparrow_cost_t()
    rc = _lib.sparrow_cost_model(_by(args), _by(cost))
    if check:
        _check(rc, "sparrow_cost_model")
    return {k: getattr(cost, k) for k, _ in sparrow_cost_t._fields_}


def sparrow_budget_tokens(sched, L: int) -> int:
    return _lib.sparrow_budget_tokens(_by(sched), L)


def sparrow_k_pages(sched, L: int) -> int:
    return _lib.sparrow_k_pages(_by(sched), L)


def sparrow_forced_count(sched, L: int) -> int:
    return _lib.sparrow_forced_count(_by(sched), L)


def sparrow_sel_count(sched, L: int) -> int:
    return _lib.sparrow_sel_count(_by(sched), L)


def sparrow_max_sel_pages(sched, max_len: int) -> int:
    return _lib.sparrow_max_sel_pages(_by(sched), max_len)


def sparrow_summarize(k_cache, summaries, page_ids, n_valid, n_update: int, shape, stream=None, *, check=True):
    rc = _lib.sparrow_summarize(_ptr(k_cache), _ptr(summaries), _ptr(page_ids), _ptr(n_valid), n_update, _by(shape), _stream(stream))
    if check:
        _check(rc, "sparrow_summarize")
    return rc


def sparrow_select(q, summaries, page_table, seq_lens, sched, sel_pages, max_sel: int, sel_count, scores_dbg,
                   workspace, shape, stream=None, *, check=True):
    rc = _lib.sparrow_select(_ptr(q), _ptr(summaries), _ptr(page_table), _ptr(seq_lens), _by(sched), _ptr(sel_pages), max_sel,
                             _ptr(sel_count), _ptr(scores_dbg), _ptr(workspace),
                             0 if workspace is None else workspace.numel() * workspace.element_size(), _by(shape), _stream(stream))
    if check:
        _check(rc, "sparrow_select")
    return rc


def sparrow_select_static_bytes() -> int:
    return _lib.sparrow_select_static_bytes()


def sparrow_select_static(q, summaries, page_table, seq_lens, sched, sel_pages, max_sel: int, sel_count, scores_dbg,
                          shape, stream=None, *, check=True):
    """sparrow_select without a workspace argument: the scratch is a fixed 4 MiB array inside the library, for callers that
    cannot allocate device memory themselves (see include/sparrow.h for the limit and the sharing rule)."""
    rc = _lib.sparrow_select_static(_ptr(q), _ptr(summaries), _ptr(page_table), _ptr(seq_lens), _by(sched), _ptr(sel_pages),
                                    max_sel, _ptr(sel_count), _ptr(scores_dbg), _by(shape), _stream(stream))
    if check:
        _check(rc, "sparrow_select_static")
    return rc


def sparrow_sparse_decode(q, k_cache, v_cache, page_table, seq_lens, sel_pages, max_sel: int, sel_count, out, lse,
                          sm_scale: float, workspace, shape, stream=None, *, check=True):
    rc = _lib.sparrow_sparse_decode(_ptr(q), _ptr(k_cache), _ptr(v_cache), _ptr(page_table), _ptr(seq_lens), _ptr(sel_pages),
                                    max_sel, _ptr(sel_count), _ptr(out), _ptr(lse), sm_scale, _ptr(workspace),
                                    0 if workspace is None else workspace.numel() * workspace.element_size(), _by(shape), _stream(stream))
    if check:
        _check(rc, "sparrow_sparse_decode")
    return rc


def sparrow_dense_decode(q, k_cache, v_cache, page_table, seq_lens, out, lse, sm_scale: float, workspace, shape,
                         stream=None, *, check=True):
    rc = _lib.sparrow_dense_decode(_ptr(q), _ptr(k_cache), _ptr(v_cache), _ptr(page_table), _ptr(seq_lens), _ptr(out), _ptr(lse),
                                   sm_scale, _ptr(workspace),
                                   0 if workspace is None else workspace.numel() * workspace.element_size(), _by(shape), _stream(stream))
    if check:
        _check(rc, "sparrow_dense_decode")
    return rc


def sparrow_append(k_new, v_new, k_cache, v_cache, summaries, page_table, seq_lens, shape, stream=None, *, check=True):
    rc = _lib.sparrow_append(_ptr(k_new), _ptr(v_new), _ptr(k_cache), _ptr(v_cache), _ptr(summaries), _ptr(page_table),
                             _ptr(seq_lens), _by(shape), _stream(stream))
    if check:
        _check(rc, "sparrow_append")
    return rc


def sparrow_step_host_block_bytes(shape):
    """(bytes of the pinned host block, offset of seq_lens, offset of page_ids, offset of n_valid)."""
    o = [_sz(0), _sz(0), _sz(0)]
    n = _lib.sparrow_step_host_block_bytes(_by(shape), _by(o[0]), _by(o[1]), _by(o[2]))
    return n, o[0].value, o[1].value, o[2].value


class HostBlock:
    """The pinned host block of sparrow_step_host as torch views (marshalling only): .q [n][Hq][128] bf16, .seq_lens [n],
    .page_ids [n], .n_valid [n] int32 all alias .block."""

    def __init__(self, shape):
        n, o_l, o_i, o_v = sparrow_step_host_block_bytes(shape)
        self.block = torch.zeros((n,), dtype=torch.uint8).pin_memory()
        ns = shape.n_seq
        self.q = self.block[: ns * shape.n_q_heads * 256].view(torch.bfloat16).view(ns, shape.n_q_heads, 128)
        self.seq_lens = self.block[o_l: o_l + 4 * ns].view(torch.int32)
        self.page_ids = self.block[o_i: o_i + 4 * ns].view(torch.int32)
        self.n_valid = self.block[o_v: o_v + 4 * ns].view(torch.int32)


def sparrow_step_host(in_block, n_update: int, has_n_valid: bool, k_cache, v_cache, summaries,
                      page_table, sched, max_sel: int, sm_scale: float, out_host, scratch, shape, stream=None, *, check=True,
                      wait=True):
    """wait=False: sparrow_step_host_async -- the step stays enqueued on the stream; synchronise before reading out_host."""
    rc = (_lib.sparrow_step_host if wait else _lib.sparrow_step_host_async)(_ptr(in_block, cuda=False), n_update, 1 if has_n_valid else 0, _ptr(k_cache), _ptr(v_cache),
                                _ptr(summaries), _ptr(page_table), _by(sched), max_sel, sm_scale, _ptr(out_host, cuda=False),
                                _ptr(scratch), scratch.numel() * scratch.element_size(), _by(shape), _stream(stream))
    if check:
        _check(rc, "sparrow_step_host")
    return rc
