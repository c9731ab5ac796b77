#!/usr/bin/env python
"""bench.py -- sparse decode-attention throughput of libsparrow_b200 on synthetic Qwen3-shaped rollouts.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--workload cfg2] [--impl sparrow|reference]

A "step" is one pass of the whole hot path over one batch: summarize the pages that just filled
-> fused score + top-k select -> split-K sparse decode + LSE merge.  Inputs are resident in HBM when the timed
region starts (`value`); `e2e` repeats the measurement through the host-buffer C-ABI entry (sparrow_step_host) with
the H2D / D2H copies inside the timed region.  One JSON line is printed by rank 0.  N > 1: replicas only, no
data-path collective (each rank its own batch and page pool; weak scaling).

`--impl reference` times the fp64 CPU oracle (as it stands, on the host cores) on a bounded sample of the same
workload: it is a deliberately slow checker, a reported baseline and not the target.
"""
from __future__ import annotations

import argparse
import json
import os
import subprocess
import sys
import threading
import time

ROOT = os.path.dirname(os.path.abspath(__file__))
sys.path.insert(0, ROOT)

import numpy as np  # noqa: E402
import torch  # noqa: E402

from paper_2606_08446_b200 import dist as D  # noqa: E402
from paper_2606_08446_b200 import workloads as W  # noqa: E402

METRIC = "sparse decode-attn tokens/s"
UNIT = "tokens/s"
KV_TILE_BYTES = 2 * 16 * 128 * 2        # K + V of one (page, kv-head): 8 KiB
SUMMARY_BYTES = 2 * 128 * 2             # min + max of one (page, kv-head): 512 B


def measured_peaks():
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(p):
        d = json.load(open(p))
        return float(d["hbm_gbs"]), "measured (MEASURED_PEAKS.json hbm_gbs, copy bandwidth)"
    return 6650.0, "fallback (B200_PROFILING.md 6.65 TB/s)"


class ClockSampler:
    """nvidia-smi clocks + throttle reasons sampled DURING the timed region."""
    Q = ("clocks.sm,clocks.max.sm,clocks_event_reasons.hw_slowdown,clocks_event_reasons.hw_thermal_slowdown,"
         "clocks_event_reasons.sw_thermal_slowdown,clocks_event_reasons.sw_power_cap")

    def __init__(self, index: int):
        self.rows, self.proc, self.index = [], None, index

    def start(self):
        try:
            self.proc = subprocess.Popen(["nvidia-smi", f"--id={self.index}", f"--query-gpu={self.Q}", "--format=csv,noheader,nounits", "-lms", "20"],
                                         stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
            self.th = threading.Thread(target=self._read, daemon=True)
            self.th.start()
        except Exception:
            self.proc = None

    def _read(self):
        for line in self.proc.stdout:
            self.rows.append(line.strip())

    def stop(self) -> dict:
        if self.proc is None:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        time.sleep(0.06)
        self.proc.terminate()
        try:
            self.proc.wait(timeout=2)
        except Exception:
            self.proc.kill()
        sm, mx, reasons = [], [], set()
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        for r in self.rows:
            f = [x.strip() for x in r.split(",")]
            if len(f) < 6:
                continue
            try:
                sm.append(float(f[0])); mx.append(float(f[1]))
            except ValueError:
                continue
            for n, v in zip(names, f[2:6]):
                if v.lower().startswith("active"):
                    reasons.add(n)
        return {"sm_mhz": float(np.median(sm)) if sm else None, "sm_max_mhz": max(mx) if mx else None,
                "reasons": sorted(reasons), "samples": len(sm)}


def algorithmic_bytes(wl, eng, lens, cnt):
    """Bytes the method itself must move per step: selected K/V tiles, candidate summaries,
    page-table / index traffic, q / out.  Returned per kernel."""
    n_pages = -(-lens // 16)
    forced = np.array([W_forced(eng, int(L)) for L in lens])
    dense_seq = cnt >= n_pages
    cand = np.where(dense_seq, 0, n_pages - forced)
    qo = wl.n_seq * wl.Hq * 128 * 2
    decode = int(cnt.sum()) * wl.Hkv * KV_TILE_BYTES + int(cnt.sum()) * wl.Hkv * 4 + int(cnt.sum()) * 4 + 2 * qo
    select = int(cand.sum()) * wl.Hkv * (SUMMARY_BYTES if getattr(eng, "landmark", "minmax") == "minmax" else SUMMARY_BYTES // 2) + int(cand.sum()) * 4 + int(cnt.sum()) * wl.Hkv * 4 + qo
    dense = int(n_pages.sum()) * wl.Hkv * KV_TILE_BYTES + int(n_pages.sum()) * 4 + 2 * qo
    return dict(decode=decode, select=select, dense=dense, sel_tiles=int(cnt.sum()) * wl.Hkv, cand_tiles=int(cand.sum()) * wl.Hkv)


def W_forced(eng, L):
    from paper_2606_08446_b200 import binding as B
    return B.sparrow_forced_count(eng.sched, L)


def time_oracle_sample(wl, h, budget_s=12.0):
    """The oracle as it stands on the host cores, on a bounded sample of sequences of the same batch."""
    import oracle
    sched = oracle.Schedule.from_spec(wl.schedule)
    n_try, best = 2, None
    while True:
        idx = np.arange(min(n_try, wl.n_seq))
        t0 = time.perf_counter()
        oracle.sparse_step(np.ascontiguousarray(h["q"][idx]), h["k_cache"], h["v_cache"], np.ascontiguousarray(h["page_table"][idx]),
                           np.ascontiguousarray(h["seq_lens"][idx]), sched, wl.sm_scale)
        dt = time.perf_counter() - t0
        best = (len(idx), dt)
        if len(idx) >= wl.n_seq or dt * 2.2 > budget_s:
            break
        n_try = min(wl.n_seq, max(n_try + 1, int(n_try * min(4.0, budget_s / max(dt, 1e-3) / 2.2))))
    # the whole batch fits the budget many times over: repeat the step for ~10 s of CPU work and take the mean
    if best[0] >= wl.n_seq and best[1] < budget_s / 4:
        reps = int(min(200, max(2, (budget_s * 0.8) // max(best[1], 1e-3))))
        idx = np.arange(wl.n_seq)
        sub = (np.ascontiguousarray(h["q"][idx]), h["k_cache"], h["v_cache"], np.ascontiguousarray(h["page_table"][idx]),
               np.ascontiguousarray(h["seq_lens"][idx]))
        t0 = time.perf_counter()
        for _ in range(reps):
            oracle.sparse_step(*sub, sched, wl.sm_scale)
        best = (wl.n_seq, (time.perf_counter() - t0) / reps)
    return best[0], best[1], oracle.num_threads()


def run_reference(args, rank):
    """--impl reference: the CPU oracle arm (rank 0 only)."""
    if rank != 0:
        return
    import oracle
    wl = W.make_config(args.workload, device="cuda" if torch.cuda.is_available() else "cpu")
    h = wl.host()
    sched = oracle.Schedule.from_spec(wl.schedule)
    # bounded sample: as many sequences as keep one step near ~1.5 s, so steps+warmup end within a few minutes
    n_s, dt, cores = time_oracle_sample(wl, h, budget_s=3.0)
    idx = np.arange(n_s)
    sub = (np.ascontiguousarray(h["q"][idx]), h["k_cache"], h["v_cache"], np.ascontiguousarray(h["page_table"][idx]),
           np.ascontiguousarray(h["seq_lens"][idx]))
    for _ in range(min(args.warmup, 2)):
        oracle.sparse_step(*sub, sched, wl.sm_scale)
    t0 = time.perf_counter()
    for _ in range(args.steps):
        oracle.sparse_step(*sub, sched, wl.sm_scale)
    dt = (time.perf_counter() - t0) / args.steps
    val = n_s / dt
    line = {"impl": "reference", "metric": METRIC, "value": val, "unit": UNIT, "n_gpus": args.gpus, "steps": args.steps,
            "warmup": args.warmup, "ms_per_step": dt * 1e3, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
            "dtype": "f64", "data": "synthetic",
            "config": {"workload": args.workload, "n_seq_sampled": int(n_s), "n_seq": wl.n_seq, "Hq": wl.Hq, "Hkv": wl.Hkv},
            "cpu_baseline": {"value": val, "unit": UNIT, "cores": cores, "kind": "oracle",
                             "sample": f"first {n_s} of {wl.n_seq} sequences of {args.workload}, full select + sparse attention per step"},
            "e2e": {"value": val, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0}, "gpu_launches": 0}
    print(json.dumps(line), flush=True)


def run_cfg4(args, rank, local_rank, world, dev):
    """BASELINE.json config 4: the 36-layer decode step at Qwen3-8B shape, batch 256, log-normal lengths; layers 0-1 dense,
    the other 34 select + sparse decode with their own q; one layer's K/V pool is ~13 GiB, so the 36 layers are mapped
    onto `--pools` rotating pools (each 100x the L2: reuse across layers adds no cache hits).  A step = all 36 layers."""
    from paper_2606_08446_b200 import binding as B
    from paper_2606_08446_b200.engine import SparrowEngine
    spec = W.CONFIGS["cfg4"]
    n_layers, n_dense, n_pools = spec["n_layers"], spec["dense_layers"], args.pools
    base_seed = D.replica_seed(4000, rank)
    wl0 = W.make_config("cfg4", seed=base_seed, device=dev)
    lens_list = wl0.seq_lens.cpu().tolist()
    wls = [wl0] + [W.make_config("cfg4", seed=base_seed + 100 * p, device=dev, lengths=("list", lens_list)) for p in range(1, n_pools)]
    st = torch.cuda.Stream(device=dev)
    engs, upds = [], []
    with torch.cuda.stream(st):
        for wl in wls:
            eng = SparrowEngine(wl)
            eng.summarize_all(stream=st)
            engs.append(eng)
            upds.append(tuple(t.to(dev) for t in W.just_filled_updates(wl)))
    st.synchronize()
    lens = np.array(lens_list)

    def layer_step(layer, count=None):
        eng, upd = engs[layer % n_pools], upds[layer % n_pools]
        n = 0
        if upd[0].numel() > 0:
            eng.summarize(upd[0], upd[1], stream=st); n += B.sparrow_last_launch_count()
        if layer < n_dense:
            eng.dense_decode(stream=st); n += B.sparrow_last_launch_count()
        else:
            eng.select(stream=st); n += B.sparrow_last_launch_count()
            eng.sparse_decode(stream=st); n += B.sparrow_last_launch_count()
        return n

    def full_step():
        return sum(layer_step(l) for l in range(n_layers))

    K, Wm = args.steps, args.warmup
    launches = 0
    with torch.cuda.stream(st):
        for _ in range(Wm):
            full_step()
        st.synchronize(); D.barrier(); torch.cuda.synchronize()
        clocks = ClockSampler(local_rank); clocks.start()
        t0, t1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        t0.record(st)
        for _ in range(K):
            launches += full_step()
        t1.record(st)
        st.synchronize(); torch.cuda.synchronize(); D.barrier()
        clk = clocks.stop()
        # per-call durations of the sparse layers (pass B, events between the calls)
        evs = []
        for l in range(n_dense, n_layers):
            eng = engs[l % n_pools]
            e = [torch.cuda.Event(enable_timing=True) for _ in range(3)]
            e[0].record(st); eng.select(stream=st); e[1].record(st); eng.sparse_decode(stream=st); e[2].record(st)
            evs.append(e)
        d0, d1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        d0.record(st)
        for l in range(n_layers):
            engs[l % n_pools].dense_decode(stream=st)
        d1.record(st)
        st.synchronize()
        # the same 36-layer step as one CUDA graph
        g = torch.cuda.CUDAGraph()
        with torch.cuda.graph(g, stream=st):
            full_step()
        g.replay(); st.synchronize()
        g0, g1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        g0.record(st)
        for _ in range(K):
            g.replay()
        g1.record(st); st.synchronize()
    total_ms = t0.elapsed_time(t1)
    value, t_max = D.whole_job_throughput(wl0.n_seq * K, total_ms * 1e-3, device=dev)
    sel_ms = float(np.mean([e[0].elapsed_time(e[1]) for e in evs]))
    dec_ms = float(np.mean([e[1].elapsed_time(e[2]) for e in evs]))
    dense_ms_all = d0.elapsed_time(d1)
    graph_ms = g0.elapsed_time(g1) / K

    # end to end: every layer through the host-buffer entry (H2D q + lens, D2H out, stream wait per layer)
    scr = [torch.zeros((B.sparrow_step_scratch_bytes(e.shape, e.max_sel),), dtype=torch.uint8, device=dev) for e in engs]
    q_h = [wl.q.cpu().pin_memory() for wl in wls]
    lens_h = wl0.seq_lens.cpu().pin_memory()
    ids_h = [u[0].cpu().pin_memory() for u in upds]; nv_h = [u[1].cpu().pin_memory() for u in upds]
    out_h = torch.empty_like(q_h[0]).pin_memory()
    dense_spec = B.make_schedule(W._sched("dense", 0, 0))

    def host_full_step():
        for l in range(n_layers):
            p = l % n_pools
            e, wl = engs[p], wls[p]
            n_upd = int(ids_h[p].numel())
            B.sparrow_step_host(q_h[p], lens_h, ids_h[p] if n_upd else None, nv_h[p] if n_upd else None, n_upd, wl.k_cache, wl.v_cache,
                                e.summaries, wl.page_table, dense_spec if l < n_dense else e.sched, e.max_sel, wl.sm_scale, out_h,
                                scr[p], e.shape, st)
    host_full_step()
    D.barrier(); torch.cuda.synchronize()
    Ke = max(1, min(K, 3))
    h0, h1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    h0.record(st)
    for _ in range(Ke):
        host_full_step()
    h1.record(st); st.synchronize()
    e2e_value, _ = D.whole_job_throughput(wl0.n_seq * Ke, h0.elapsed_time(h1) * 1e-3, device=dev)
    if rank != 0:
        return
    eng = engs[0]
    cnt = eng.sel_count.cpu().numpy()
    ab = algorithmic_bytes(wl0, eng, lens, cnt)
    peak, peak_src = measured_peaks()
    dec_gbs = ab["decode"] / (dec_ms * 1e-3) / 1e9
    sel_gbs = ab["select"] / (sel_ms * 1e-3) / 1e9
    qbytes = int(q_h[0].numel() * 2)
    line = {
        "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": K, "warmup": Wm, "ms_per_step": t_max * 1e3 / K,
        "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "bf16", "data": "synthetic",
        "config": {"workload": "cfg4", "n_seq": wl0.n_seq, "Hq": wl0.Hq, "Hkv": wl0.Hkv, "head_dim": 128, "page_size": 16,
                   "n_layers": n_layers, "dense_layers": n_dense, "kv_pools": n_pools, "len_min": int(lens.min()), "len_max": int(lens.max()),
                   "len_median": float(np.median(lens)), "schedule": wl0.schedule["kind"], "selected_pages_per_seq_mean": float(cnt.mean()),
                   "parallelism": f"replicas x{world} (no collective)",
                   "l2": "inputs larger than L2: each layer streams %.0f MB from its own ~13 GiB pool" % ((ab["decode"] + ab["select"]) / 1e6),
                   "timing": "a step = 36 layers (2 dense + 34 select + sparse decode) over rotating K/V pools; value from K steps between two events"},
        "roofline": {"bound": "hbm", "kernel": "decode_kernel<sparse> (mean over the 34 sparse layers, events between the calls)",
                     "achieved": dec_gbs, "peak": peak, "unit": "GB/s", "frac": dec_gbs / peak, "traffic": None, "peak_source": peak_src,
                     "algorithmic_bytes_per_launch": ab["decode"], "avg_launch_ms": dec_ms, "frac_of_8TBs_nominal": dec_gbs / 8000.0},
        "kernels": {"select": {"ms": sel_ms, "algorithmic_bytes": ab["select"], "achieved_GBs": sel_gbs, "frac": sel_gbs / peak},
                    "sparse_decode": {"ms": dec_ms, "algorithmic_bytes": ab["decode"], "achieved_GBs": dec_gbs, "frac": dec_gbs / peak},
                    "dense_decode_all_layers": {"ms": dense_ms_all, "achieved_GBs": n_layers * ab["dense"] / (dense_ms_all * 1e-3) / 1e9}},
        "graph_ms_per_step": graph_ms,
        "dense_tokens_per_s": wl0.n_seq / (dense_ms_all * 1e-3),
        "speedup_vs_dense": dense_ms_all / (t_max * 1e3 / K),
        "e2e": {"value": e2e_value, "unit": UNIT, "h2d_bytes_per_step": n_layers * (qbytes + int(lens_h.numel() * 4)),
                "d2h_bytes_per_step": n_layers * qbytes},
        "gpu_launches": launches, "clocks": clk,
        "paper_context": "Sparrow rollout speedup 2.0x for Qwen3-8B on 4xH200 (PAPER.md:7; whole-engine, not this kernel path)",
    }
    print(json.dumps(line), flush=True)


def run_table4(args, rank, dev):
    """PAPER.md:426-434 (Table 4): sparse decode at KV budget 1024 tokens with page sizes 16 / 32 / 64 / 128 (configs
    16-64, 32-32, 64-16, 128-8) and 16k / 24k / 32k tokens of past KV, Qwen3-1.7B attention shape, batch 16.  The paper
    times a full-model decode pass on one H200 (4.1-5.4 ms, flat in the page size); this times the attention path of
    ONE layer (select + sparse decode) on the B200, where the page size only changes the summary stream."""
    if rank != 0:
        return
    from paper_2606_08446_b200.engine import SparrowEngine
    rows = []
    for past in (16384, 24576, 32768):
        for page in (16, 32, 64, 128):
            sched = W._sched("fixed", 64, 512, fixed_tokens=1024)
            wl = W.make_workload("table4", n_seq=16, Hq=16, Hkv=8, lengths=("list", [past] * 16), schedule=sched, plant=True,
                                 seed=4400 + page, device=dev, page_size=page)
            eng = SparrowEngine(wl)
            eng.summarize_all()
            res = {}
            for name, fn in (("select", eng.select), ("sparse_decode", eng.sparse_decode), ("dense_decode", eng.dense_decode)):
                for _ in range(3):
                    fn()
                best = 1e9
                for _ in range(3):
                    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
                    e0.record()
                    for _ in range(args.steps):
                        fn()
                    e1.record(); torch.cuda.synchronize()
                    best = min(best, e0.elapsed_time(e1) * 1e3 / args.steps)
                res[name] = best
            rows.append({"past_kv": past, "page_size": page, "pages_kept": int(eng.sel_count[0].item()),
                         "select_us": res["select"], "sparse_decode_us": res["sparse_decode"],
                         "sparse_us": res["select"] + res["sparse_decode"], "dense_decode_us": res["dense_decode"]})
            del eng, wl
            torch.cuda.empty_cache()
    print(json.dumps({"table4": rows, "unit": "us per layer (attention path only)", "steps": args.steps,
                      "config": {"workload": "table4", "n_seq": 16, "Hq": 16, "Hkv": 8, "budget_tokens": 1024, "sink_tokens": 64,
                                 "local_tokens": 512},
                      "paper_context": "Table 4 (PAPER.md:426-434): full-model decode pass 4.13-5.41 ms on 1xH200, flat in page size"}),
          flush=True)


def run_acceptance(args, rank, dev):
    """throughput of sparrow_acceptance (alpha per position + per-bin 5-percentile) on synthetic top-20
    lists shaped like the paper's study (37K-token trajectories, 2K bins -> 19 bins)."""
    if rank != 0:
        return
    from paper_2606_08446_b200 import binding as B
    inp = W.make_acceptance_inputs(96, 37000, top_n=20, seed=3, device=dev)
    n_pos, n_bins = int(inp["positions"].numel()), 19
    alpha = torch.zeros((n_pos,), dtype=torch.float32, device=dev)
    bq = torch.zeros((n_bins,), dtype=torch.float32, device=dev)
    bc = torch.zeros((n_bins,), dtype=torch.int32, device=dev)
    ws = torch.zeros((B.sparrow_acceptance_workspace_bytes(n_bins),), dtype=torch.uint8, device=dev)
    call = lambda: B.sparrow_acceptance(inp["ids_p"], inp["logp_p"], inp["ids_q"], inp["logp_q"], inp["positions"], 20, 2048, n_bins,
                                        0.05, alpha, bq, bc, ws)
    for _ in range(3):
        call()
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    e0.record()
    for _ in range(args.steps):
        call()
    e1.record(); torch.cuda.synchronize()
    ms = e0.elapsed_time(e1) / args.steps
    peak, peak_src = measured_peaks()
    alg = n_pos * (4 * 20 * 4 + 4) + 3 * n_pos * 8          # lists in, alpha out; three selection passes over (alpha, position)
    print(json.dumps({"metric": "acceptance-rate positions/s", "value": n_pos / (ms * 1e-3), "unit": "positions/s", "ms_per_call": ms,
                      "steps": args.steps, "config": {"workload": "acceptance", "n_pos": n_pos, "top_n": 20, "n_bins": n_bins, "bin_tokens": 2048},
                      "roofline": {"bound": "hbm", "achieved": alg / (ms * 1e-3) / 1e9, "peak": peak, "unit": "GB/s",
                                   "frac": alg / (ms * 1e-3) / 1e9 / peak, "peak_source": peak_src, "algorithmic_bytes_per_call": alg,
                                   "note": "7 launches per call; the alpha kernel (80 % of the time) is issue-bound, not HBM-bound: ncu sm__throughput 93 %, "
                                           "214 warp instructions per position, DRAM 19 % of peak"},
                      "bin_count": bc.cpu().tolist(), "bin_5pct": [round(float(x), 4) for x in bq.cpu().tolist()]}), flush=True)


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=30)
    ap.add_argument("--warmup", type=int, default=5)
    ap.add_argument("--workload", default="cfg2", choices=list(W.CONFIGS))
    ap.add_argument("--pools", type=int, default=4, help="cfg4 only: distinct K/V pools the 36 layers rotate over (~14 GiB each)")
    ap.add_argument("--impl", default="sparrow", choices=["sparrow", "reference"])
    ap.add_argument("--step-form", default="two-launches", choices=["two-launches", "fused"],
                    help="select + sparse decode as two launches (default, measured faster) or as the one cooperative sparrow_step launch")
    ap.add_argument("--table4", action="store_true", help="page-size sweep at budget 1024 (PAPER.md Table 4) instead of the step benchmark")
    ap.add_argument("--acceptance", action="store_true", help="time sparrow_acceptance (SURVEY 8(f)-3) instead of the step benchmark")
    ap.add_argument("--landmark", default="minmax", choices=["minmax", "mean"],
                    help="page landmark: per-channel min/max (north_star's default, 512 B) or the mean key (the paper's cost model, 256 B)")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-check", action="store_true", help="skip the sampled oracle self-check before timing")
    args = ap.parse_args()
    args.warmup = max(args.warmup, 3)
    if args.landmark == "mean":
        args.no_cpu_baseline = True      # the timed CPU baseline is the default (min/max) path's oracle

    rank, local_rank, world = D.env_world()
    if args.impl == "reference":
        run_reference(args, rank)
        return
    assert torch.cuda.is_available(), "bench.py needs a CUDA device: there is no CPU fallback"
    torch.cuda.set_device(local_rank)
    dev = torch.device("cuda", local_rank)
    D.init("nccl")
    if args.table4:
        run_table4(args, rank, dev)
        return
    if args.acceptance:
        run_acceptance(args, rank, dev)
        return
    if args.workload == "cfg4":
        run_cfg4(args, rank, local_rank, world, dev)
        return
    from paper_2606_08446_b200 import binding as B
    from paper_2606_08446_b200.engine import SparrowEngine

    base_seed = 1000 * int("".join(ch for ch in args.workload if ch.isdigit()) or 0)
    wl = W.make_config(args.workload, seed=D.replica_seed(base_seed, rank), device=dev)
    eng = SparrowEngine(wl, landmark=args.landmark)
    st = torch.cuda.Stream(device=dev)
    upd = tuple(t.to(dev) for t in W.just_filled_updates(wl))
    with torch.cuda.stream(st):
        eng.summarize_all(stream=st)
        t_sum0, t_sum1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        t_sum0.record(st); eng.summarize_all(stream=st); t_sum1.record(st)
    st.synchronize()
    bulk_sum_ms = t_sum0.elapsed_time(t_sum1)
    n_bulk = int(eng._ids.numel())

    lens = wl.seq_lens.cpu().numpy()
    # ---- correctness gate before timing (rank 0, a few sampled sequences) ----
    h = None
    if rank == 0 and not args.no_check:
        sys.path.insert(0, os.path.join(ROOT, "tests"))
        from parity_util import check_sparse_step
        with torch.cuda.stream(st):
            eng.step(updates=upd, stream=st)
        st.synchronize()
        h = wl.host()
        idx = sorted({int(lens.argmin()), int(lens.argmax()), 0})
        chk = check_sparse_step(eng, wl, h=h, idx=idx)
    else:
        chk = None

    fused = args.step_form == "fused"

    def one_step():
        n = 0
        if upd[0].numel() > 0:
            eng.summarize(upd[0], upd[1], stream=st); n += B.sparrow_last_launch_count()
        if fused:
            return n
        eng.select(stream=st); n += B.sparrow_last_launch_count()
        return n

    def attend():
        """second half of the step: the sparse decode launch (or the whole fused select + decode launch)"""
        if fused:
            eng.fused_step(stream=st)
        else:
            eng.sparse_decode(stream=st)
        return B.sparrow_last_launch_count()

    # ---- timed region: K steps, device-resident inputs, events on the launching stream ----
    # Region A (-> `value`): K whole steps back to back, one event before and one after, as a caller runs them.
    # Region B (-> `roofline`, `kernels`): the same K steps again with an event between the calls, which gives each
    # kernel's launch duration; the extra event records cost a few microseconds per step, so B is not the
    # throughput number.
    K, Wm = args.steps, args.warmup
    ev = [[torch.cuda.Event(enable_timing=True) for _ in range(4)] for _ in range(K)]
    launches = 0
    clocks = ClockSampler(local_rank); clocks.start()      # nvidia-smi needs tens of ms to come up: started before the warm-up
    with torch.cuda.stream(st):
        for _ in range(Wm):
            one_step(); attend()
        st.synchronize()
        D.barrier()
        torch.cuda.synchronize()
        t_beg = torch.cuda.Event(enable_timing=True); t_end = torch.cuda.Event(enable_timing=True)
        t_beg.record(st)
        for k in range(K):
            launches += one_step()
            launches += attend()
        t_end.record(st)
        st.synchronize()
        torch.cuda.synchronize()
        D.barrier()
        for k in range(K):
            ev[k][3].record(st)
            if upd[0].numel() > 0:
                eng.summarize(upd[0], upd[1], stream=st)
            ev[k][0].record(st)
            if not fused:
                eng.select(stream=st)
            ev[k][1].record(st)
            attend()
            ev[k][2].record(st)
        st.synchronize()
    total_ms = t_beg.elapsed_time(t_end)
    sum_ms = float(np.mean([e[3].elapsed_time(e[0]) for e in ev]))
    sel_ms = float(np.mean([e[0].elapsed_time(e[1]) for e in ev]))
    dec_ms = float(np.mean([e[1].elapsed_time(e[2]) for e in ev]))
    value, t_max = D.whole_job_throughput(wl.n_seq * K, total_ms * 1e-3, device=dev)

    # ---- dense path of the same library on the same inputs (speedup denominator) ----
    Kd = max(3, min(K, 10))
    with torch.cuda.stream(st):
        for _ in range(2):
            eng.dense_decode(stream=st)
        d0, d1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        d0.record(st)
        for _ in range(Kd):
            eng.dense_decode(stream=st)
        d1.record(st)
    st.synchronize()
    dense_ms = d0.elapsed_time(d1) / Kd

    # ---- end to end through the host-buffer C-ABI entry (H2D + D2H inside the timed region) ----
    scratch = torch.zeros((B.sparrow_step_scratch_bytes(eng.shape, eng.max_sel),), dtype=torch.uint8, device=dev)
    q_h, lens_h = wl.q.cpu().pin_memory(), wl.seq_lens.cpu().pin_memory()
    ids_h, nv_h = upd[0].cpu().pin_memory(), upd[1].cpu().pin_memory()
    out_h = torch.empty_like(q_h).pin_memory()
    n_upd = int(ids_h.numel())

    def host_step():
        B.sparrow_step_host(q_h, lens_h, ids_h if n_upd else None, nv_h if n_upd else None, n_upd, wl.k_cache, wl.v_cache,
                            eng.summaries, wl.page_table, eng.sched, eng.max_sel, wl.sm_scale, out_h, scratch, eng.shape, st)
    for _ in range(Wm):
        host_step()
    D.barrier(); torch.cuda.synchronize()
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    e0.record(st)
    for _ in range(K):
        host_step()
    e1.record(st); st.synchronize()
    # The timed loops of this run last a few ms each and nvidia-smi samples every 20 ms: keep the same kernels running
    # (untimed) until the sampler has a few readings under this load.
    t_wait = time.perf_counter()
    while len(clocks.rows) < 4 and time.perf_counter() - t_wait < 3.0:
        with torch.cuda.stream(st):
            for _ in range(50):
                one_step(); attend()
        st.synchronize()
    clk = clocks.stop()
    e2e_value, _ = D.whole_job_throughput(wl.n_seq * K, e0.elapsed_time(e1) * 1e-3, device=dev)
    h2d = int(q_h.numel() * 2 + lens_h.numel() * 4 + n_upd * 8)
    d2h = int(out_h.numel() * 2)
    e2e_match = bool(torch.equal(out_h, eng.out.cpu()))

    if rank != 0:
        return
    cnt = eng.sel_count.cpu().numpy()
    ab = algorithmic_bytes(wl, eng, lens, cnt)
    peak, peak_src = measured_peaks()
    roof_bytes = ab["decode"] + (ab["select"] if fused else 0)       # fused: one launch streams the summaries too
    roof_kernel = ("step_kernel (one sparrow_step call: scoring + top-k + decode + LSE merge)" if fused else
                   "decode_kernel<sparse> (one sparrow_sparse_decode call; LSE merge fused in the same launch)")
    dec_gbs = roof_bytes / (dec_ms * 1e-3) / 1e9
    sel_gbs = ab["select"] / (sel_ms * 1e-3) / 1e9
    dense_gbs = ab["dense"] / (dense_ms * 1e-3) / 1e9
    traffic = None      # dram__bytes_read.sum + dram__bytes_write.sum of the decode kernel from the committed ncu capture
    tp = os.path.join(ROOT, "profiles", "ncu_traffic.txt")
    if os.path.exists(tp):
        for ln in open(tp):
            f = ln.split()
            if len(f) >= 3 and f[0] == args.workload and f[1] == ("step_kernel" if fused else "decode_kernel"):
                traffic = int(f[2])

    line = {
        "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": K, "warmup": Wm,
        "ms_per_step": t_max * 1e3 / K, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
        "dtype": "bf16", "data": "synthetic",
        "config": {"workload": args.workload, "n_seq": wl.n_seq, "Hq": wl.Hq, "Hkv": wl.Hkv, "head_dim": 128, "page_size": 16,
                   "len_min": int(lens.min()), "len_max": int(lens.max()), "schedule": wl.schedule["kind"], "step_form": args.step_form, "landmark": args.landmark,
                   "sink_tokens": wl.schedule["sink_tokens"], "local_tokens": wl.schedule["local_tokens"],
                   "selected_pages_per_seq_mean": float(cnt.mean()), "parallelism": f"replicas x{world} (no collective)",
                   "l2": "inputs larger than L2: %.0f MB touched per step vs 126 MB L2" % ((ab["decode"] + ab["select"]) / 1e6),
                   "timing": "value: K steps back to back between two events; roofline/kernels: a second pass of K steps with an event between the calls"},
        "roofline": {"bound": "hbm", "kernel": roof_kernel,
                     "achieved": dec_gbs, "peak": peak, "unit": "GB/s", "frac": dec_gbs / peak, "traffic": traffic,
                     "peak_source": peak_src, "algorithmic_bytes_per_launch": roof_bytes, "avg_launch_ms": dec_ms,
                     "frac_of_8TBs_nominal": dec_gbs / 8000.0},
        "kernels": {"summarize_step": {"ms": sum_ms, "pages": int(upd[0].numel())},
                    "select": {"ms": sel_ms, "algorithmic_bytes": ab["select"], "achieved_GBs": sel_gbs, "frac": sel_gbs / peak},
                    "sparse_decode": {"ms": dec_ms, "algorithmic_bytes": ab["decode"], "achieved_GBs": dec_gbs, "frac": dec_gbs / peak},
                    "dense_decode": {"ms": dense_ms, "algorithmic_bytes": ab["dense"], "achieved_GBs": dense_gbs, "frac": dense_gbs / peak},
                    "bulk_summarize": {"ms": bulk_sum_ms, "pages": n_bulk,
                                       "achieved_GBs": n_bulk * wl.Hkv * (4096 + 512) / (bulk_sum_ms * 1e-3) / 1e9}},
        "sparse_path_GBs": (ab["decode"] + ab["select"]) / (t_max / K) / 1e9,
        "dense_tokens_per_s": wl.n_seq / (dense_ms * 1e-3),
        "speedup_vs_dense": dense_ms / (t_max * 1e3 / K),
        "ideal_speedup_bytes_ratio": ab["dense"] / (ab["decode"] + ab["select"]),
        "e2e": {"value": e2e_value, "unit": UNIT, "h2d_bytes_per_step": h2d, "d2h_bytes_per_step": d2h,
                "matches_device_path": e2e_match},
        "gpu_launches": launches,
        "clocks": clk,
        "paper_context": "Sparrow rollout speedups 2.2x/2.4x/2.0x for Qwen3-1.7B/4B/8B on 4xH200 (PAPER.md:7; whole-engine, not this kernel path)",
    }
    if chk is not None:
        line["self_check"] = {"sampled_seqs": len(idx), **{k: chk[k] for k in ("units", "differing_units", "max_abs", "mean_abs", "lse_max_abs")}}
    if not args.no_cpu_baseline:
        h = h or wl.host()
        n_s, dt, cores = time_oracle_sample(wl, h)
        line["cpu_baseline"] = {"value": n_s / dt, "unit": UNIT, "cores": cores, "kind": "oracle",
                                "sample": f"first {n_s} of {wl.n_seq} sequences of {args.workload}: full select + sparse-attention steps, {dt:.3f} s each (mean over ~10 s of CPU work when one step is short)"}
    print(json.dumps(line), flush=True)


if __name__ == "__main__":
    main()
