"""Timelines of the select and decode kernels from the TRACING build of the library (csrc/common.cuh, -DSPARROW_TRACE).

    python -m paper_2606_08446_b200.trace select cfg2 [cfg5 cfg3]     per-CTA phases + resident / streaming / top-k counts over time
    python -m paper_2606_08446_b200.trace decode cfg5 [cfg2 cfg3]     ramp, per-warp exits, spread of the CTA ends
    python -m paper_2606_08446_b200.trace gaps   cfg5 [cfg2]          select -> decode -> select on one stream: overlap and gaps

The kernels of the tracing build write %globaltimer stamps (one 64-bit store per stamp, thread 0 or lane 0 only); the
arithmetic is the normal build's.  The stamps cost ~1 us per launch, so launch TIMES are taken from the normal build
(bench.py); this tool is for where inside a launch the time goes.  The reports under profiles/ name the command that made
them.  Needs a GPU; there is no CPU path.
"""
from __future__ import annotations

import os
import sys

_HERE = os.path.dirname(os.path.abspath(__file__))
_TRACE_LIB = os.path.join(_HERE, "libsparrow_b200_trace.so")
os.environ["SPARROW_B200_LIB"] = _TRACE_LIB          # before binding is imported
if not os.path.exists(_TRACE_LIB):
    from . import build as _bld
    _bld.build(trace=True)

import numpy as np  # noqa: E402
import torch  # noqa: E402

from . import binding as B  # noqa: E402
from . import workloads as W  # noqa: E402
from .engine import SparrowEngine  # noqa: E402

SLOTS, DEC_CTA, DEC_WARP, DEC_WARPS = 65536, 60000, 56000, 9


def _setup(cfg):
    wl = W.make_config(cfg, seed=1000 * int("".join(ch for ch in cfg if ch.isdigit())), device="cuda")
    eng = SparrowEngine(wl)
    eng.summarize_all()
    for _ in range(5):
        eng.select()
        eng.sparse_decode()
    torch.cuda.synchronize()
    return wl, eng


def _us(x):
    return np.asarray(x, dtype=np.float64) / 1e3


def trace_select(cfg):
    wl, eng = _setup(cfg)
    tr = torch.zeros((SLOTS, 8), dtype=torch.int64, device="cuda")
    B.sparrow_trace_set(tr)
    eng.sparse_decode()
    eng.select()                       # follows a decode launch and is followed by one, as in the step
    eng.sparse_decode()
    torch.cuda.synchronize()
    B.sparrow_trace_set(None)
    t = tr.cpu().numpy()[:DEC_WARP]
    t = t[t[:, 0] > 0].astype(np.float64)
    t0 = t[:, 0].min()
    end = np.where(t[:, 5] > 0, t[:, 5], np.where(t[:, 4] > 0, t[:, 4], np.where(t[:, 3] > 0, t[:, 3], t[:, 1])))
    work, last = t[:, 2] > 0, t[:, 5] > 0
    med = lambda x: float(np.median(_us(x)))
    print(f"select {cfg}: {len(t)} CTAs, {int(work.sum())} with pages to score, {int(last.sum())} ran a unit's top-k; "
          f"first CTA start -> last CTA end {_us(end.max() - t0):.1f} us")
    print(f"  medians: prologue {med(t[work, 1] - t[work, 0]):.2f} us | summary stream {med(t[work, 2] - t[work, 1]):.2f} us "
          f"(p90 {np.percentile(_us(t[work, 2] - t[work, 1]), 90):.2f}) | barrier + arrival atomic {med(t[work, 4] - t[work, 2]):.2f} us | "
          f"top-k {med(t[last, 5] - t[last, 4]):.2f} us (max {_us(t[last, 5] - t[last, 4]).max():.2f})")
    L = t[last]
    print(f"  top-k split: keys -> shared + min / max {med(L[:, 7] - L[:, 4]):.2f} us | radix passes {med(L[:, 6] - L[:, 7]):.2f} us | "
          f"compaction {med(L[:, 5] - L[:, 6]):.2f} us")
    print("  t us   resident streaming topk")
    span = _us(end.max() - t0)
    for lo in np.arange(0.0, span + 2.0, 2.0):
        inb = lambda a, b: int(((_us(a - t0) < lo + 2) & (_us(b - t0) > lo)).sum())
        print(f"  {lo:5.0f}   {inb(t[:, 0], end):7d} {inb(t[work, 1], t[work, 2]):9d} {inb(t[last, 4], t[last, 5]):4d}")


def _decode_rows(tr):
    t = tr.cpu().numpy()
    cta = t[DEC_CTA:DEC_CTA + 148].astype(np.float64)
    warp = t[DEC_WARP:DEC_WARP + 148 * DEC_WARPS].reshape(148, DEC_WARPS, 8).astype(np.float64)
    return cta, warp


def trace_decode(cfg):
    wl, eng = _setup(cfg)
    for rep in range(2):
        tr = torch.zeros((SLOTS, 8), dtype=torch.int64, device="cuda")
        eng.select()
        torch.cuda.synchronize()
        B.sparrow_trace_set(tr)
        eng.sparse_decode()
        torch.cuda.synchronize()
        B.sparrow_trace_set(None)
        cta, warp = _decode_rows(tr)
        t0 = cta[:, 0].min()
        row = lambda name, x: print(f"  {name:34s} min {x.min():7.2f}  median {np.median(x):7.2f}  max {x.max():7.2f}")
        print(f"decode {cfg} (run {rep}): us after the first CTA's first instruction, over the 148 CTAs")
        row("dependency wait over", _us(cta[:, 1] - t0))
        row("prefix table built", _us(cta[:, 2] - t0))
        row("first tile landed", _us(cta[:, 4] - t0))
        row("look-up warp finished", _us(cta[:, 3] - t0))
        ex = _us(warp[:, :, 1] - t0)
        cons = np.sort(ex[:, :8], axis=1)
        row("first consumer warp out", cons[:, 0])
        row("7th consumer warp out", cons[:, 6])
        row("last consumer warp out = CTA end", cons[:, 7])
        pct = np.percentile(cons[:, 7], [0, 10, 50, 90, 100])
        print("  CTA ends, percentiles 0 / 10 / 50 / 90 / 100: " + " / ".join(f"{x:.1f}" for x in pct))
    del eng, wl


def trace_gaps(cfg):
    wl, eng = _setup(cfg)
    for order in ("select->decode", "decode->select"):
        tr = torch.zeros((SLOTS, 8), dtype=torch.int64, device="cuda")
        eng.select()
        eng.sparse_decode()
        torch.cuda.synchronize()
        B.sparrow_trace_set(tr)
        if order == "select->decode":
            eng.select()
            eng.sparse_decode()
        else:
            eng.sparse_decode()
            eng.select()
        torch.cuda.synchronize()
        B.sparrow_trace_set(None)
        t = tr.cpu().numpy()
        s = t[:DEC_WARP]
        s = s[s[:, 0] > 0].astype(np.float64)
        cta, warp = _decode_rows(tr)
        s0, s1 = s[:, 0].min(), s[:, 1:6].max()
        d0, d_go, d1 = cta[:, 0].min(), cta[:, 1].min(), warp[:, :, 1].max()
        if order == "select->decode":
            print(f"{cfg} {order}: select {_us(s1 - s0):.1f} us | decode CTAs resident {_us(s1 - d0):.1f} us before select ends, released "
                  f"{_us(d_go - s1):.1f} us after it | decode {_us(d1 - d_go):.1f} us | pair {_us(d1 - s0):.1f} us")
        else:
            print(f"{cfg} {order}: decode {_us(d1 - d0):.1f} us | gap to select's first CTA {_us(s0 - d1):.1f} us | select {_us(s1 - s0):.1f} us | "
                  f"pair {_us(s1 - d0):.1f} us")


def main(argv):
    if len(argv) < 2 or argv[0] not in ("select", "decode", "gaps"):
        print(__doc__)
        return 2
    assert torch.cuda.is_available(), "trace.py needs a CUDA device"
    fn = {"select": trace_select, "decode": trace_decode, "gaps": trace_gaps}[argv[0]]
    for cfg in argv[1:]:
        fn(cfg)
        torch.cuda.empty_cache()
    return 0


if __name__ == "__main__":
    sys.exit(main(sys.argv[1:]))
