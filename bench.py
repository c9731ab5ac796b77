#!/usr/bin/env python
"""bench.py -- sparse decode-attention throughput of libsparrow_b200 on synthetic Qwen3-shaped rollouts.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--workload cfg4|cfg2|cfg3|cfg5] [--impl sparrow|reference]

A "step" is one pass of the whole hot path over one batch: summarize the pages that just filled
-> fused score + top-k select -> split-K sparse decode + LSE merge.  The default workload is BASELINE.json config 4,
the largest single-GPU configuration (BASELINE.json's `metric` names no config): one step = the 36-layer decode step
at Qwen3-8B shape, batch 256 (layers 0-1 dense, 34 sparse) over rotating K/V pools.  The same JSON line carries a
`per_config` block with the single-layer configs 2, 3 and 5.  Inputs are resident in HBM when the timed region starts
(`value`); `e2e` repeats the measurement through the host-buffer C-ABI entry (sparrow_step_host) with the H2D / D2H
copies inside the timed region.  One JSON line is printed by rank 0.  N > 1: replicas only, no data-path collective
(each rank its own batch and page pool; weak scaling); without a torchrun environment `--gpus N` starts the N ranks
itself.

`--impl reference` times the fp64 CPU oracle (as it stands, on the host cores) on a bounded sample of the same
workload: it is a deliberately slow checker, a reported baseline and not the target.
Other modes: --rollout T, --table4 (8(f)-2), --acceptance (8(f)-3).
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
MIN_KERNEL_SAMPLES = 50                 # >= 50 timed launches behind every per-kernel figure
PAPER_CONTEXT = ("Sparrow rollout speedups 2.2x/2.4x/2.0x for Qwen3-1.7B/4B/8B on 4xH200 (PAPER.md:7; whole-engine, "
                 "not this kernel path)")


def measured_peaks():
    """(HBM GB/s, bf16 FLOP/s, where from).  The roofline denominator is the driver-measured copy bandwidth."""
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(p):
        d = json.load(open(p))
        return float(d["hbm_gbs"]), float(d.get("bf16_tflops", 1590.0)) * 1e12, "measured (MEASURED_PEAKS.json hbm_gbs, copy bandwidth)"
    return 6650.0, 1.59e15, "fallback (B200_PROFILING.md 6.65 TB/s)"


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


def same_result(a, b, deterministic: bool):
    """Two decodes of the same inputs (host-buffer entry vs device path): (max abs difference, agree?).  With
    SPARROW_FLAG_DETERMINISTIC they must be bit-equal.  Otherwise the tiles are handed out at run time and the two agree to
    the arithmetic's own error: 2^-7 relative (a few bf16 steps of the larger value) + 1.5e-3 absolute per element -- the
    tolerance of tests/parity_util.assert_same_result, not a fixed max-abs (one bf16 step at |out| >= 0.5 is already 3.9e-3)."""
    a, b = a.float(), b.float()
    d = (a - b).abs()
    if deterministic:
        return float(d.max()), bool(torch.equal(a, b))
    tol = 2.0 ** -7 * torch.maximum(a.abs(), b.abs()) + 1.5e-3
    return float(d.max()), bool((d <= tol).all())


def stats_ms(xs) -> dict:
    xs = np.asarray(xs, dtype=np.float64)
    return {"ms": float(xs.mean()), "ms_median": float(np.median(xs)), "ms_min": float(xs.min()), "samples": int(xs.size)}


def block_ms(fn, n, st) -> float:
    """Mean duration of ONE call of fn: n calls back to back on stream st between two events (no event, and so no idle
    gap, between the calls -- the way the step runs them)."""
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    fn()
    e0.record(st)
    for _ in range(n):
        fn()
    e1.record(st)
    st.synchronize()
    return e0.elapsed_time(e1) / n


def algorithmic_bytes(wl, eng, lens, cnt):
    """Bytes the method itself must move per step: selected K/V tiles, candidate summaries,
    page-table / index traffic, q / out.  Returned per kernel."""
    from paper_2606_08446_b200 import binding as B
    n_pages = -(-lens // 16)
    forced = np.array([B.sparrow_forced_count(eng.sched, int(L)) for L in lens])
    dense_seq = cnt >= n_pages
    cand = np.where(dense_seq, 0, n_pages - forced)
    qo = wl.n_seq * wl.Hq * 128 * 2
    lm_bytes = SUMMARY_BYTES if getattr(eng, "landmark", "minmax") == "minmax" else SUMMARY_BYTES // 2
    decode = int(cnt.sum()) * wl.Hkv * KV_TILE_BYTES + int(cnt.sum()) * wl.Hkv * 4 + int(cnt.sum()) * 4 + 2 * qo
    select = int(cand.sum()) * wl.Hkv * lm_bytes + int(cand.sum()) * 4 + int(cnt.sum()) * wl.Hkv * 4 + qo
    dense = int(n_pages.sum()) * wl.Hkv * KV_TILE_BYTES + int(n_pages.sum()) * 4 + 2 * qo
    return dict(decode=decode, select=select, dense=dense, sel_tiles=int(cnt.sum()) * wl.Hkv, cand_tiles=int(cand.sum()) * wl.Hkv)


def ncu_traffic(workload: str, kernel: str):
    """dram__bytes_read.sum + dram__bytes_write.sum per launch of `kernel` on `workload` from the committed ncu capture
    (profiles/ncu_traffic.txt).  Returns (bytes or None, note): None when there is no capture of THIS build -- a line
    is valid only for the kernel sources it was measured on (their hash is stored beside it)."""
    from paper_2606_08446_b200 import build as bld
    tp = os.path.join(ROOT, "profiles", "ncu_traffic.txt")
    if not os.path.exists(tp):
        return None, "no profiles/ncu_traffic.txt"
    here = bld.source_hash()
    stale = None
    for ln in open(tp):
        f = ln.split()
        if len(f) >= 4 and not ln.startswith("#") and f[0] == workload and f[1] == kernel:
            if f[3] == here:
                return int(f[2]), f"ncu --set full capture of this build (source hash {here})"
            stale = f[3]
    if stale:
        return None, f"the committed capture is of another build (source hash {stale}, this build {here})"
    return None, "no capture for this workload"


def cost_model_block(wl, eng, lens, cnt, hbm_gbs, flops) -> dict:
    """the paper's cost model (Eq. 2-3, App. F :474-498) evaluated by
    sparrow_cost_model for ONE decode step of every sequence of the batch (L_in = L - 1 cached tokens, L_out = 1, budget
    K = 16 x the pages the schedule keeps), attention terms only (P = 0), at the B200's intensity I = flops per bf16
    element moved; summed over the batch -> predicted dense / sparse cost ratio, to be read beside the measured one."""
    from paper_2606_08446_b200 import binding as B
    r = wl.Hq // wl.Hkv
    intensity = flops / (hbm_gbs * 1e9 / 2.0)
    out = {"intensity_flop_per_elem": intensity}
    for c in (1.0, 2.0):
        dense = sparse = 0.0
        for L, k in zip(lens.tolist(), cnt.tolist()):
            cm = B.sparrow_cost_model(params=0.0, batch_size=1.0, n_samples=1.0, L_in=float(L - 1), L_out=1.0, D=128.0 * wl.Hkv,
                                      r=float(r), intensity=intensity, budget_tokens=float(16 * k), page_size=16.0, landmarks_per_page=c)
            dense += cm["dense_total"]
            sparse += cm["sparse_total"]
        out[f"predicted_dense_over_sparse_c{int(c)}"] = dense / sparse
    out["note"] = ("c1 = one landmark vector per page (the paper's model), c2 = this library's min/max pair (R1); per-step form of "
                   "Eq. 2-3: L_in = L - 1, L_out = 1, P = 0")
    return out


def time_oracle(wl, h, idx, budget_s=10.0, dense=True):
    """The oracle as it stands on the host cores, on the sequences `idx` of the batch (h = a host view that holds them):
    seconds per sparse step (select + sparse attention) and per dense-attention step."""
    import oracle
    sys.path.insert(0, os.path.join(ROOT, "tests"))
    from parity_util import sub_host
    hs = sub_host(h, idx)
    sched = oracle.Schedule.from_spec(wl.schedule)
    args = (hs["q"], hs["k_cache"], hs["v_cache"], hs["page_table"], hs["seq_lens"])
    t0 = time.perf_counter()
    oracle.sparse_step(*args, sched, wl.sm_scale)
    dt = time.perf_counter() - t0
    reps = int(min(200, max(1, (budget_s * 0.6) // max(dt, 1e-3))))
    if reps > 1:
        t0 = time.perf_counter()
        for _ in range(reps):
            oracle.sparse_step(*args, sched, wl.sm_scale)
        dt = (time.perf_counter() - t0) / reps
    dt_dense = None
    if dense:
        t0 = time.perf_counter()
        oracle.dense_step(*args, wl.sm_scale)
        dt_dense = time.perf_counter() - t0
    return dt, dt_dense, oracle.num_threads()


def oracle_sample_size(wl, target_s=1.5, n_total=None) -> int:
    """How many of the first sequences keep one oracle sparse step near target_s: the first two are timed and the
    count is scaled linearly (the oracle's cost is linear in the number of sequences)."""
    import oracle
    h = W.host_subset(wl, [0, 1] if wl.n_seq > 1 else [0])
    sched = oracle.Schedule.from_spec(wl.schedule)
    for _ in range(2):                                   # the first call pays the library load and the thread pool start
        t0 = time.perf_counter()
        oracle.sparse_step(h["q"], h["k_cache"], h["v_cache"], h["page_table"], h["seq_lens"], sched, wl.sm_scale)
        dt = max(time.perf_counter() - t0, 1e-4)
    return max(2, min(n_total or wl.n_seq, int(len(h["seq_lens"]) * target_s / dt)))


# ---------------------------------------------------------------------------------------------------------------
def run_reference(args, rank):
    """--impl reference: the CPU oracle arm (rank 0 only), same config / metric / unit as the library's arm.  Each step
    is a bounded sample of the workload: the first n_s sequences (cfg4: of ONE layer pool -- one sparse layer and one
    dense layer timed per step, the 36-layer step = 34 x sparse + 2 x dense)."""
    if rank != 0:
        return
    import oracle
    dev = "cuda" if torch.cuda.is_available() else "cpu"
    cfg = args.workload
    spec = W.CONFIGS[cfg]
    seed = 1000 * int("".join(ch for ch in cfg if ch.isdigit()) or 0)
    if dev == "cpu" and cfg in ("cfg3", "cfg4"):
        # no GPU to draw a 10+ GiB pool with: draw only the sampled sequences (same length law, same value law)
        g = torch.Generator().manual_seed(seed)
        lens_all = W.draw_lengths(spec["lengths"], spec["n_seq"], g)
        n_total = spec["n_seq"]
        probe = W.make_config(cfg, seed=seed, device=dev, n_seq=2, lengths=("list", lens_all[:2]))
        n_s = min(oracle_sample_size(probe, target_s=1.5, n_total=n_total), 32)     # bounded: the pool is drawn on the CPU here
        wl = W.make_config(cfg, seed=seed, device=dev, n_seq=n_s, lengths=("list", lens_all[:n_s]))
    else:
        wl = W.make_config(cfg, seed=seed, device=dev)
        n_total = wl.n_seq
        n_s = oracle_sample_size(wl, target_s=1.5)
    idx = list(range(min(n_s, wl.n_seq)))
    h = W.host_subset(wl, idx)
    sched = oracle.Schedule.from_spec(wl.schedule)
    sub = (h["q"], h["k_cache"], h["v_cache"], h["page_table"], h["seq_lens"])
    n_layers, n_dense = spec.get("n_layers", 1), spec.get("dense_layers", 0)

    def one_step():
        t0 = time.perf_counter()
        oracle.sparse_step(*sub, sched, wl.sm_scale)
        t1 = time.perf_counter()
        if n_dense:
            oracle.dense_step(*sub, wl.sm_scale)
        t2 = time.perf_counter()
        return (n_layers - n_dense) * (t1 - t0) + n_dense * (t2 - t1)      # seconds of the whole (multi-layer) step on the sample
    for _ in range(min(args.warmup, 2)):
        one_step()
    dts = [one_step() for _ in range(args.steps)]
    dt = float(np.mean(dts))
    val = len(idx) / dt
    what = (f"first {len(idx)} of {n_total} sequences of {cfg}" +
            (f", one layer pool: each step times one sparse layer (select + sparse attention) and one dense layer, "
             f"step time = {n_layers - n_dense} x sparse + {n_dense} x dense" if n_layers > 1 else ": full select + sparse attention per step"))
    line = {"impl": "reference", "metric": METRIC, "value": val, "unit": UNIT, "n_gpus": args.gpus, "steps": args.steps,
            "warmup": args.warmup, "ms_per_step": dt * 1e3, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
            "dtype": "f64", "data": "synthetic",
            "config": {"workload": cfg, "n_seq": n_total, "Hq": wl.Hq, "Hkv": wl.Hkv, "head_dim": 128, "page_size": 16,
                       "n_layers": n_layers, "dense_layers": n_dense, "n_seq_sampled": len(idx)},
            "cpu_baseline": {"value": val, "unit": UNIT, "cores": oracle.num_threads(), "kind": "oracle", "sample": what},
            "e2e": {"value": val, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0}, "gpu_launches": 0}
    print(json.dumps(line), flush=True)


# ---------------------------------------------------------------------------------------------------------------
def self_check(eng, wl, idx, dense_idx=None) -> dict:
    """Oracle check of a step that has already run on `eng` (selection + summaries + out / lse on the sequences idx;
    the dense entry on dense_idx), on a compacted host copy of just those sequences' pages."""
    sys.path.insert(0, os.path.join(ROOT, "tests"))
    from parity_util import check_dense, check_sparse_step
    idx = sorted(set(int(i) for i in idx))
    h = W.host_subset(wl, idx)
    st = check_sparse_step(eng, wl, h=h, idx=idx)
    res = {"seqs": len(idx), **{k: st[k] for k in ("units", "differing_units", "band_pages", "max_abs", "mean_abs", "lse_max_abs")}}
    if dense_idx:
        sd = check_dense(eng, wl, h=h, idx=sorted(set(int(i) for i in dense_idx)))
        res["dense_seqs"] = len(set(dense_idx)); res["dense_max_abs"] = sd["max_abs"]; res["dense_lse_max_abs"] = sd["lse_max_abs"]
    return res, h


def run_single(args, cfg, rank, local_rank, world, dev, headline=True) -> dict:
    """One single-layer configuration (cfg2 / cfg3 / cfg5): the step = summarize(just filled) -> select -> sparse decode."""
    from paper_2606_08446_b200 import binding as B
    from paper_2606_08446_b200.engine import SparrowEngine
    base_seed = 1000 * int("".join(ch for ch in cfg if ch.isdigit()) or 0)
    wl = W.make_config(cfg, seed=D.replica_seed(base_seed, rank), device=dev)
    wl_chk = wl                                          # the packed arrays: what the oracle checks and times against
    if args.kv_layout == "nhd":                          # the same values in [page][token][kv-head][128] pools (sparrow_shape_t kv_stride_*)
        import copy
        wl = copy.copy(wl)
        wl.k_cache = wl_chk.k_cache.permute(0, 2, 1, 3).contiguous()
        wl.v_cache = wl_chk.v_cache.permute(0, 2, 1, 3).contiguous()
    eng = SparrowEngine(wl, landmark=args.landmark, kv_layout=args.kv_layout, deterministic=args.deterministic)
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

    # ---- correctness gate before timing (rank 0): every sequence of cfg2 / cfg5, 16 of cfg3 ----
    chk, h = None, None
    if rank == 0 and not args.no_check:
        with torch.cuda.stream(st):
            eng.step(updates=upd, stream=st)
            eng.dense_decode(stream=st)
        st.synchronize()
        ext = [int(lens.argmin()), int(lens.argmax())]
        others = [i for i in np.random.default_rng(2).permutation(wl.n_seq).tolist() if i not in ext]
        idx = list(range(wl.n_seq)) if wl.n_seq <= 64 else ext + others[:16 - len(set(ext))]
        chk, h = self_check(eng, wl_chk, idx, dense_idx=ext)

    def one_step():
        n = 0
        if upd[0].numel() > 0:
            eng.summarize(upd[0], upd[1], stream=st); n += B.sparrow_last_launch_count()
        eng.select(stream=st); n += B.sparrow_last_launch_count()
        return n

    def attend():
        """second half of the step: the sparse decode launch"""
        eng.sparse_decode(stream=st)
        return B.sparrow_last_launch_count()

    # ---- timed region: K steps, device-resident inputs, events on the launching stream ----
    # Region A (-> `value`): K whole steps back to back, one event before and one after, as a caller runs them.
    # Region B (-> `roofline`, `kernels`): max(K, 50) more steps with an event between the calls, which gives each kernel's
    # launch duration (mean, median and min); the extra event records cost a few microseconds per step, so B is not the
    # throughput number.
    K, Wm = args.steps, args.warmup
    KB = max(K, MIN_KERNEL_SAMPLES)
    ev = [[torch.cuda.Event(enable_timing=True) for _ in range(4)] for _ in range(KB)]
    launches = 0
    clocks = ClockSampler(local_rank)
    if headline:
        clocks.start()      # nvidia-smi needs tens of ms to come up: started before the warm-up
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
        for k in range(KB):
            ev[k][3].record(st)
            if upd[0].numel() > 0:
                eng.summarize(upd[0], upd[1], stream=st)
            ev[k][0].record(st)
            eng.select(stream=st)
            ev[k][1].record(st)
            attend()
            ev[k][2].record(st)
        st.synchronize()
    total_ms = t_beg.elapsed_time(t_end)
    k_sum = stats_ms([e[3].elapsed_time(e[0]) for e in ev])
    k_sel = stats_ms([e[0].elapsed_time(e[1]) for e in ev])
    k_dec = stats_ms([e[1].elapsed_time(e[2]) for e in ev])
    # Region C (-> the `ms` behind `roofline` and `kernels`): KB launches of ONE kernel back to back between two events.  The
    # bracketed samples of region B carry an event record on each side of every launch (~2 us of idle stream each on these
    # 40-100 us kernels); they are kept as median / min.
    for k_, fn_ in ((k_sel, lambda: eng.select(stream=st)), (k_dec, attend)):
        with torch.cuda.stream(st):
            k_["ms_bracketed"] = k_["ms"]
            k_["ms"] = block_ms(fn_, KB, st)
    value, t_max = D.whole_job_throughput(wl.n_seq * K, total_ms * 1e-3, device=dev)

    # ---- dense path of the same library on the same inputs (speedup denominator) ----
    Kd = max(3, min(K, 10))
    with torch.cuda.stream(st):
        for _ in range(2):
            eng.dense_decode(stream=st)
        evd = [torch.cuda.Event(enable_timing=True) for _ in range(Kd + 1)]
        evd[0].record(st)
        for i in range(Kd):
            eng.dense_decode(stream=st)
            evd[i + 1].record(st)
    st.synchronize()
    k_dense = stats_ms([evd[i].elapsed_time(evd[i + 1]) for i in range(Kd)])
    dense_ms = evd[0].elapsed_time(evd[Kd]) / Kd

    # ---- end to end through the host-buffer C-ABI entry (ONE H2D of the packed input block + D2H inside the timed region) ----
    scratch = torch.zeros((B.sparrow_step_scratch_bytes(eng.shape, eng.max_sel),), dtype=torch.uint8, device=dev)
    hb = B.HostBlock(eng.shape)
    hb.q.copy_(wl.q.cpu()); hb.seq_lens.copy_(wl.seq_lens.cpu())
    n_upd = int(upd[0].numel())
    hb.page_ids[:n_upd] = upd[0].cpu(); hb.n_valid[:n_upd] = upd[1].cpu()
    out_h = torch.empty_like(hb.q).pin_memory()

    def host_step():
        B.sparrow_step_host(hb.block, n_upd, False, wl.k_cache, wl.v_cache, eng.summaries, wl.page_table, eng.sched, eng.max_sel,
                            wl.sm_scale, out_h, scratch, eng.shape, st)
    for _ in range(Wm):
        host_step()
    D.barrier(); torch.cuda.synchronize()
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    e0.record(st)
    for _ in range(K):
        host_step()
    e1.record(st); st.synchronize()
    clk = None
    if headline:
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
    h2d = int(hb.q.numel() * 2 + hb.seq_lens.numel() * 4 + n_upd * 4)
    d2h = int(out_h.numel() * 2)
    # The tiles are handed to the consumer warps at run time, so the running maximum under which a probability is rounded
    # to bf16 -- and the fp32 summation order -- differ from call to call: two calls agree to the arithmetic's own error
    # (the oracle gate on max-abs is 3e-3), not bit for bit.
    e2e_diff, e2e_match = same_result(out_h, eng.out.cpu(), args.deterministic)

    if rank != 0:
        return {}
    cnt = eng.sel_count.cpu().numpy()
    ab = algorithmic_bytes(wl, eng, lens, cnt)
    peak, flops, peak_src = measured_peaks()
    roof_bytes = ab["decode"]
    roof_kernel = "decode_kernel<sparse> (one sparrow_sparse_decode call; LSE merge fused in the same launch)"
    gbs = lambda b, ms: b / (ms * 1e-3) / 1e9
    dec_gbs, sel_gbs, dense_gbs = gbs(roof_bytes, k_dec["ms"]), gbs(ab["select"], k_sel["ms"]), gbs(ab["dense"], dense_ms)
    traffic, traffic_note = ncu_traffic(cfg, "decode_kernel" + ("@deterministic" if args.deterministic else ""))
    ms_step = t_max * 1e3 / K
    res = {
        "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": K, "warmup": Wm,
        "ms_per_step": ms_step, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
        "dtype": "bf16", "data": "synthetic",
        "config": {"workload": cfg, "n_seq": wl.n_seq, "Hq": wl.Hq, "Hkv": wl.Hkv, "head_dim": 128, "page_size": 16,
                   "len_min": int(lens.min()), "len_max": int(lens.max()), "schedule": wl.schedule["kind"], "landmark": args.landmark,
                   "kv_layout": args.kv_layout, "deterministic": bool(args.deterministic),
                   "sink_tokens": wl.schedule["sink_tokens"], "local_tokens": wl.schedule["local_tokens"],
                   "selected_pages_per_seq_mean": float(cnt.mean()), "parallelism": f"replicas x{world} (no collective)",
                   "l2": "inputs larger than L2: %.0f MB touched per step vs 126 MB L2" % ((ab["decode"] + ab["select"]) / 1e6),
                   "timing": f"value: K steps back to back between two events; roofline/kernels: ms = {KB} launches of the one kernel back to back between two events; "
                             f"ms_bracketed / ms_median / ms_min = {KB} more steps with an event between the calls"},
        "roofline": {"bound": "hbm", "kernel": roof_kernel,
                     "achieved": dec_gbs, "peak": peak, "unit": "GB/s", "frac": dec_gbs / peak, "traffic": traffic, "traffic_note": traffic_note,
                     "peak_source": peak_src, "algorithmic_bytes_per_launch": roof_bytes, "avg_launch_ms": k_dec["ms"],
                     "median_launch_ms": k_dec["ms_median"], "min_launch_ms": k_dec["ms_min"], "frac_of_8TBs_nominal": dec_gbs / 8000.0,
                     "frac_of_read_stream": dec_gbs / dense_gbs,
                     "read_stream_note": "the copy peak is not a ceiling for a read-only stream: the library's dense entry on the same inputs reaches "
                                         "%.0f GB/s; frac_of_read_stream = achieved / that" % dense_gbs},
        "kernels": {"summarize_step": {**k_sum, "pages": int(upd[0].numel())},
                    "select": {**k_sel, "algorithmic_bytes": ab["select"], "achieved_GBs": sel_gbs, "frac": sel_gbs / peak,
                               "frac_of_8TBs_nominal": sel_gbs / 8000.0},
                    "sparse_decode": {**k_dec, "algorithmic_bytes": ab["decode"], "achieved_GBs": dec_gbs, "frac": dec_gbs / peak,
                                      "frac_of_8TBs_nominal": dec_gbs / 8000.0},
                    "dense_decode": {**k_dense, "algorithmic_bytes": ab["dense"], "achieved_GBs": dense_gbs, "frac": dense_gbs / peak},
                    "bulk_summarize": {"ms": bulk_sum_ms, "pages": n_bulk,
                                       "achieved_GBs": n_bulk * wl.Hkv * (4096 + 512) / (bulk_sum_ms * 1e-3) / 1e9}},
        "sparse_path_GBs": (ab["decode"] + ab["select"]) / (t_max / K) / 1e9,
        "sparse_path_frac": (ab["decode"] + ab["select"]) / (t_max / K) / 1e9 / peak,
        "dense_tokens_per_s": wl.n_seq / (dense_ms * 1e-3),
        "speedup_vs_dense": dense_ms / ms_step,
        "ideal_speedup_bytes_ratio": ab["dense"] / (ab["decode"] + ab["select"]),
        "cost_model": cost_model_block(wl, eng, lens, cnt, peak, flops),
        "e2e": {"value": e2e_value, "unit": UNIT, "h2d_bytes_per_step": h2d, "d2h_bytes_per_step": d2h,
                "matches_device_path": e2e_match, "max_abs_vs_device_path": e2e_diff, "frac_of_device_value": e2e_value / value},
        "gpu_launches": launches,
    }
    if clk is not None:
        res["clocks"] = clk
        res["paper_context"] = PAPER_CONTEXT
    if chk is not None:
        res["self_check"] = chk
    if not args.no_cpu_baseline:
        n_s = oracle_sample_size(wl_chk, target_s=1.0)
        idx = list(range(n_s))
        hh = h if (h is not None and set(idx) <= set(h["seq_index"].tolist())) else W.host_subset(wl_chk, idx)
        dt, dt_dense, cores = time_oracle(wl_chk, hh, idx)
        res["cpu_baseline"] = {"value": n_s / dt, "unit": UNIT, "cores": cores, "kind": "oracle",
                               "dense_value": n_s / dt_dense,
                               "sample": f"first {n_s} of {wl.n_seq} sequences of {cfg}: full select + sparse-attention steps, {dt:.3f} s each "
                                         f"(mean over ~6 s of CPU work when one step is short); dense attention on the same sequences {dt_dense:.3f} s"}
    del eng, wl, wl_chk, scratch
    torch.cuda.empty_cache()
    return res


def run_cfg4(args, rank, local_rank, world, dev) -> dict:
    """BASELINE.json config 4: the 36-layer decode step at Qwen3-8B shape, batch 256, log-normal lengths; layers 0-1 dense,
    the other 34 select + sparse decode; one layer's K/V pool is ~13 GiB, so the 36 layers are mapped onto `--pools`
    rotating pools with their own q, K, V and page tables (each 100x the L2: reuse across layers adds no cache hits).
    A step = all 36 layers."""
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
            eng = SparrowEngine(wl, deterministic=args.deterministic)
            eng.summarize_all(stream=st)
            engs.append(eng)
            upds.append(tuple(t.to(dev) for t in W.just_filled_updates(wl)))
    st.synchronize()
    lens = np.array(lens_list)

    def layer_step(layer):
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

    # ---- correctness gate before timing: sampled sequences of EVERY pool, a sparse layer and the dense entry ----
    chk = None
    h0 = None
    if rank == 0 and not args.no_check:
        with torch.cuda.stream(st):
            full_step()
            for e in engs:
                e.dense_decode(stream=st)
        st.synchronize()
        sys.path.insert(0, os.path.join(ROOT, "tests"))
        import oracle
        sched_o = oracle.Schedule.from_spec(wl0.schedule)
        dense_inside = [i for i in range(wl0.n_seq) if oracle.k_pages(sched_o, int(lens[i])) >= -(-int(lens[i]) // 16)]
        ext = [int(lens.argmin()), int(lens.argmax())]
        rng = np.random.default_rng(4)
        per_pool = []
        for p, (e, wl) in enumerate(zip(engs, wls)):
            must = sorted(set(ext + dense_inside[:2]))
            idx = must + [i for i in rng.permutation(wl.n_seq).tolist() if i not in must][:8 - len(must)]
            c, hh = self_check(e, wl, idx, dense_idx=ext[:1] + dense_inside[:1])
            per_pool.append(c)
            if p == 0:
                h0 = hh
        chk = {"pools": n_pools, "layers_checked": "one sparse layer and the dense entry per pool",
               "seqs": sum(c["seqs"] for c in per_pool), "units": sum(c["units"] for c in per_pool),
               "differing_units": sum(c["differing_units"] for c in per_pool), "band_pages": sum(c["band_pages"] for c in per_pool),
               "dense_in_sparse_batch_seqs_checked": len(dense_inside[:2]),
               "max_abs": max(c["max_abs"] for c in per_pool), "mean_abs": max(c["mean_abs"] for c in per_pool),
               "lse_max_abs": max(c["lse_max_abs"] for c in per_pool), "dense_max_abs": max(c["dense_max_abs"] for c in per_pool),
               "dense_lse_max_abs": max(c["dense_lse_max_abs"] for c in per_pool)}

    K, Wm = args.steps, args.warmup
    launches = 0
    clocks = ClockSampler(local_rank); clocks.start()
    with torch.cuda.stream(st):
        for _ in range(Wm):
            full_step()
        st.synchronize(); D.barrier(); torch.cuda.synchronize()
        # Region A (-> value): K 36-layer steps back to back; one event per step boundary (one record per ~22 ms) gives
        # the per-step median and min as well
        evs = [torch.cuda.Event(enable_timing=True) for _ in range(K + 1)]
        evs[0].record(st)
        for k in range(K):
            launches += full_step()
            evs[k + 1].record(st)
        st.synchronize(); torch.cuda.synchronize(); D.barrier()
        clk = clocks.stop()
        # Region B: per-call durations of the sparse layers (events between the calls), >= 50 samples of each kernel
        kev = []
        reps = -(-MIN_KERNEL_SAMPLES // (n_layers - n_dense))
        for _ in range(reps):
            for l in range(n_dense, n_layers):
                eng = engs[l % n_pools]
                e = [torch.cuda.Event(enable_timing=True) for _ in range(3)]
                e[0].record(st); eng.select(stream=st); e[1].record(st); eng.sparse_decode(stream=st); e[2].record(st)
                kev.append(e)
        dev_ev = [torch.cuda.Event(enable_timing=True) for _ in range(n_layers + 1)]
        dev_ev[0].record(st)
        for l in range(n_layers):
            engs[l % n_pools].dense_decode(stream=st)
            dev_ev[l + 1].record(st)
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
    total_ms = evs[0].elapsed_time(evs[K])
    step_stats = stats_ms([evs[k].elapsed_time(evs[k + 1]) for k in range(K)])
    value, t_max = D.whole_job_throughput(wl0.n_seq * K, total_ms * 1e-3, device=dev)
    k_sel = stats_ms([e[0].elapsed_time(e[1]) for e in kev])
    k_dec = stats_ms([e[1].elapsed_time(e[2]) for e in kev])
    # ms = launches of the one kernel back to back (rotating over the pools, as the layers do) between two events; the
    # event-bracketed samples above are kept as ms_bracketed / median / min
    n_blk = -(-MIN_KERNEL_SAMPLES // n_pools) * n_pools
    for k_, name_ in ((k_sel, "select"), (k_dec, "sparse_decode")):
        e0_, e1_ = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        with torch.cuda.stream(st):
            e0_.record(st)
            for i_ in range(n_blk):
                getattr(engs[i_ % n_pools], name_)(stream=st)
            e1_.record(st)
        st.synchronize()
        k_["ms_bracketed"] = k_["ms"]
        k_["ms"] = e0_.elapsed_time(e1_) / n_blk
    k_dense = stats_ms([dev_ev[l].elapsed_time(dev_ev[l + 1]) for l in range(n_layers)])
    dense_ms_all = dev_ev[0].elapsed_time(dev_ev[n_layers])
    graph_ms = g0.elapsed_time(g1) / K

    # ---- end to end: every layer through the host-buffer entry (one packed H2D, D2H out, stream wait per layer) ----
    scr = [torch.zeros((B.sparrow_step_scratch_bytes(e.shape, e.max_sel),), dtype=torch.uint8, device=dev) for e in engs]
    hbs = []
    for wl, upd, e in zip(wls, upds, engs):
        hb = B.HostBlock(e.shape)
        hb.q.copy_(wl.q.cpu()); hb.seq_lens.copy_(wl.seq_lens.cpu())
        n_upd = int(upd[0].numel())
        hb.page_ids[:n_upd] = upd[0].cpu(); hb.n_valid[:n_upd] = upd[1].cpu()
        hbs.append((hb, n_upd))
    out_h = torch.empty_like(hbs[0][0].q).pin_memory()
    dense_spec = B.make_schedule(W._sched("dense", 0, 0))

    def host_full_step():
        for l in range(n_layers):
            p = l % n_pools
            e, wl, (hb, n_upd) = engs[p], wls[p], hbs[p]
            B.sparrow_step_host(hb.block, n_upd, False, wl.k_cache, wl.v_cache, e.summaries, wl.page_table,
                                dense_spec if l < n_dense else e.sched, e.max_sel, wl.sm_scale, out_h, scr[p], e.shape, st,
                                wait=False)          # 36 layers enqueued (each with its H2D and D2H) ...
        st.synchronize()                                 # ... and ONE wait per step, where the caller reads the result
    host_full_step()
    D.barrier(); torch.cuda.synchronize()
    Ke = K                                               # the same K steps as the device-resident value
    h0e, h1e = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    h0e.record(st)
    for _ in range(Ke):
        host_full_step()
    h1e.record(st); st.synchronize()
    e2e_value, _ = D.whole_job_throughput(wl0.n_seq * Ke, h0e.elapsed_time(h1e) * 1e-3, device=dev)
    ref_o = engs[(n_layers - 1) % n_pools].out.cpu().float()
    e2e_diff, e2e_match = same_result(out_h, ref_o, args.deterministic)
    if rank != 0:
        return {}
    eng = engs[0]
    cnt = eng.sel_count.cpu().numpy()
    ab = algorithmic_bytes(wl0, eng, lens, cnt)
    peak, flops, peak_src = measured_peaks()
    gbs = lambda b, ms: b / (ms * 1e-3) / 1e9
    dec_gbs, sel_gbs = gbs(ab["decode"], k_dec["ms"]), gbs(ab["select"], k_sel["ms"])
    hb0 = hbs[0][0]
    qbytes = int(hb0.q.numel() * 2)
    traffic, traffic_note = ncu_traffic("cfg4", "decode_kernel" + ("@deterministic" if args.deterministic else ""))
    ms_step = t_max * 1e3 / K
    step_bytes = (n_layers - n_dense) * (ab["decode"] + ab["select"]) + n_dense * ab["dense"]
    res = {
        "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": K, "warmup": Wm, "ms_per_step": ms_step,
        "ms_per_step_median": step_stats["ms_median"], "ms_per_step_min": step_stats["ms_min"],
        "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "bf16", "data": "synthetic",
        "config": {"workload": "cfg4", "n_seq": wl0.n_seq, "Hq": wl0.Hq, "Hkv": wl0.Hkv, "head_dim": 128, "page_size": 16,
                   "n_layers": n_layers, "dense_layers": n_dense, "kv_pools": n_pools, "deterministic": bool(args.deterministic), "len_min": int(lens.min()), "len_max": int(lens.max()),
                   "len_median": float(np.median(lens)), "schedule": wl0.schedule["kind"], "selected_pages_per_seq_mean": float(cnt.mean()),
                   "parallelism": f"replicas x{world} (no collective)",
                   "l2": "inputs larger than L2: each layer streams %.0f MB from its own ~13 GiB pool" % ((ab["decode"] + ab["select"]) / 1e6),
                   "timing": "a step = 36 layers (2 dense + 34 select + sparse decode) over rotating K/V pools; value from K steps between "
                             "two events (an event per step boundary gives median / min); kernels: ms = launches of the one kernel back to back between two events, "
                             "ms_bracketed / ms_median / ms_min = a pass with an event between the calls"},
        "roofline": {"bound": "hbm", "kernel": "decode_kernel<sparse> (one sparrow_sparse_decode call; LSE merge fused in the same launch)",
                     "achieved": dec_gbs, "peak": peak, "unit": "GB/s", "frac": dec_gbs / peak, "traffic": traffic, "traffic_note": traffic_note,
                     "peak_source": peak_src, "algorithmic_bytes_per_launch": ab["decode"], "avg_launch_ms": k_dec["ms"],
                     "median_launch_ms": k_dec["ms_median"], "min_launch_ms": k_dec["ms_min"], "frac_of_8TBs_nominal": dec_gbs / 8000.0,
                     "frac_of_read_stream": dec_gbs / gbs(ab["dense"], k_dense["ms"]),
                     "read_stream_note": "the copy peak is not a ceiling for a read-only stream: the library's dense entry on the same inputs reaches "
                                         "%.0f GB/s; frac_of_read_stream = achieved / that" % gbs(ab["dense"], k_dense["ms"])},
        "kernels": {"select": {**k_sel, "algorithmic_bytes": ab["select"], "achieved_GBs": sel_gbs, "frac": sel_gbs / peak,
                               "frac_of_8TBs_nominal": sel_gbs / 8000.0},
                    "sparse_decode": {**k_dec, "algorithmic_bytes": ab["decode"], "achieved_GBs": dec_gbs, "frac": dec_gbs / peak,
                                      "frac_of_8TBs_nominal": dec_gbs / 8000.0},
                    "dense_decode": {**k_dense, "algorithmic_bytes": ab["dense"], "achieved_GBs": gbs(ab["dense"], k_dense["ms"]),
                                     "frac": gbs(ab["dense"], k_dense["ms"]) / peak}},
        "step_GBs": step_bytes / (ms_step * 1e-3) / 1e9, "step_frac": step_bytes / (ms_step * 1e-3) / 1e9 / peak,
        "graph_ms_per_step": graph_ms,
        "dense_ms_per_step": dense_ms_all,
        "dense_tokens_per_s": wl0.n_seq / (dense_ms_all * 1e-3),
        "speedup_vs_dense": dense_ms_all / ms_step,
        "ideal_speedup_bytes_ratio": n_layers * ab["dense"] / step_bytes,
        "cost_model": cost_model_block(wl0, eng, lens, cnt, peak, flops),
        "e2e": {"value": e2e_value, "unit": UNIT, "h2d_bytes_per_step": n_layers * (qbytes + int(hb0.seq_lens.numel() * 4) + 4 * hbs[0][1]),
                "d2h_bytes_per_step": n_layers * qbytes, "steps_timed": Ke, "matches_device_path": e2e_match, "max_abs_vs_device_path": e2e_diff, "frac_of_device_value": e2e_value / value},
        "gpu_launches": launches, "clocks": clk,
        "paper_context": "Sparrow rollout speedup 2.0x for Qwen3-8B on 4xH200 (PAPER.md:7; whole-engine, not this kernel path)",
    }
    if chk is not None:
        res["self_check"] = chk
    if not args.no_cpu_baseline:
        # the oracle on ONE layer pool, first n_s sequences: a sparse layer and a dense layer, scaled to the 36-layer step
        n_s = oracle_sample_size(wl0, target_s=1.5)
        idx = list(range(n_s))
        hh = W.host_subset(wl0, idx)
        dt, dt_dense, cores = time_oracle(wl0, hh, idx, budget_s=6.0)
        t_step = (n_layers - n_dense) * dt + n_dense * dt_dense
        res["cpu_baseline"] = {"value": n_s / t_step, "unit": UNIT, "cores": cores, "kind": "oracle",
                               "dense_value": n_s / (n_layers * dt_dense),
                               "sample": f"first {n_s} of {wl0.n_seq} sequences of one cfg4 layer pool: one sparse layer (select + sparse attention) "
                                         f"{dt:.3f} s and one dense layer {dt_dense:.3f} s on the host cores, scaled to the step as "
                                         f"{n_layers - n_dense} x sparse + {n_dense} x dense (BASELINE.md section 4)"}
    del engs, wls, scr
    torch.cuda.empty_cache()
    return res


# ---------------------------------------------------------------------------------------------------------------
def run_rollout(args, rank, dev):
    """SURVEY.md 8(f)-1 / PAPER.md:498 ("sparse attention avoids O(L_out^2) scaling and instead yields O(K L_out)"): a T-step
    rollout (append -> select -> sparse decode per step, lengths on the device) against the dense rollout (append -> dense
    decode) on the same growing cache, each bucket of `--rollout-bucket` steps captured as ONE CUDA graph; cumulative time
    and algorithmic bytes per bucket.  Qwen3-1.7B attention shape, batch 64, prompt 1024 tokens, budget = the paper's
    native TABLE form in 2K bins (1024 tokens up to 2K context, then +256 tokens per bin, capped at 3072)."""
    if rank != 0:
        return
    from paper_2606_08446_b200 import binding as B
    from paper_2606_08446_b200.engine import SparrowEngine
    T, bucket = args.rollout, args.rollout_bucket
    T = -(-T // bucket) * bucket
    n_seq, Hq, Hkv, L_in = 64, 16, 8, 1024
    table = tuple(min(64 + 16 * b, 192) for b in range(32))          # pages per 2K-token length bin
    sched = W._sched("table", 64, 512, table_pages=table, bin_tokens=2048)
    peak, _, peak_src = measured_peaks()
    rows = {}
    for mode in ("sparse", "dense"):
        wl = W.make_workload("rollout", n_seq=n_seq, Hq=Hq, Hkv=Hkv, lengths=("list", [L_in] * n_seq), schedule=sched, plant=True,
                             seed=6100, device=dev, reserve_tokens=T + 1)
        eng = SparrowEngine(wl)
        eng.summarize_all(); eng.reserve(T)
        qs, ks, vs = W.make_rollout_inputs(wl, bucket, seed=5)       # one bucket of step inputs, reused by every bucket
        out = torch.zeros((bucket, n_seq, Hq, 128), dtype=torch.bfloat16, device=dev)
        st = torch.cuda.Stream(device=dev)
        # eager warm-up of the kernels on a throw-away engine state is not needed: the first graph replay is the warm-up of
        # its own bucket, and a bucket cannot be replayed twice (it advances the lengths).  Module load is warmed here:
        eng.select(); eng.sparse_decode(); eng.dense_decode(); torch.cuda.synchronize()
        with torch.cuda.stream(st):
            g = torch.cuda.CUDAGraph()
            with torch.cuda.graph(g, stream=st):
                eng.rollout(qs, ks, vs, out, dense=(mode == "dense"), stream=st)
            eng.note_appended(T - bucket)                             # the captured bucket is replayed T / bucket times
            evs = [torch.cuda.Event(enable_timing=True) for _ in range(T // bucket + 1)]
            evs[0].record(st)
            for b in range(T // bucket):
                g.replay()
                evs[b + 1].record(st)
        st.synchronize()
        assert int(wl.seq_lens[0].item()) == L_in + T
        rows[mode] = [evs[b].elapsed_time(evs[b + 1]) for b in range(T // bucket)]
        del eng, wl, g
        torch.cuda.empty_cache()
    sched_c = B.make_schedule(sched)
    table_rows, cum_s, cum_d, cum_bs, cum_bd = [], 0.0, 0.0, 0, 0
    for b in range(T // bucket):
        Ls = [L_in + b * bucket + t + 1 for t in range(bucket)]
        sel_pages = sum(B.sparrow_sel_count(sched_c, L) for L in Ls)
        cand = sum(max(0, -(-L // 16) - B.sparrow_forced_count(sched_c, L)) if B.sparrow_sel_count(sched_c, L) < -(-L // 16) else 0 for L in Ls)
        all_pages = sum(-(-L // 16) for L in Ls)
        bytes_s = n_seq * Hkv * (sel_pages * KV_TILE_BYTES + cand * SUMMARY_BYTES)
        bytes_d = n_seq * Hkv * all_pages * KV_TILE_BYTES
        cum_s += rows["sparse"][b]; cum_d += rows["dense"][b]; cum_bs += bytes_s; cum_bd += bytes_d
        table_rows.append({"steps": f"{b * bucket + 1}-{(b + 1) * bucket}", "context_end": L_in + (b + 1) * bucket,
                           "budget_tokens_end": 16 * B.sparrow_k_pages(sched_c, L_in + (b + 1) * bucket),
                           "sparse_ms": rows["sparse"][b], "dense_ms": rows["dense"][b], "sparse_cum_ms": cum_s, "dense_cum_ms": cum_d,
                           "sparse_GB": bytes_s / 1e9, "dense_GB": bytes_d / 1e9, "sparse_cum_GB": cum_bs / 1e9, "dense_cum_GB": cum_bd / 1e9,
                           "sparse_us_per_step": rows["sparse"][b] * 1e3 / bucket, "dense_us_per_step": rows["dense"][b] * 1e3 / bucket})
    print(json.dumps({"rollout": table_rows, "config": {"workload": "rollout", "n_seq": n_seq, "Hq": Hq, "Hkv": Hkv, "L_in": L_in, "T": T,
                                                         "bucket_steps": bucket, "schedule": "table (2K bins): 64 + 16 b pages, cap 192; sink 64, local 512",
                                                         "graphs": "one CUDA graph per bucket (append -> select -> sparse decode, or append -> dense decode, per step)"},
                      "cumulative_speedup": cum_d / cum_s, "cumulative_bytes_ratio": cum_bd / cum_bs, "peak_GBs": peak, "peak_source": peak_src,
                      "paper_context": "PAPER.md:498: sparse attention avoids O(L_out^2) scaling and instead yields O(K L_out) memory growth"}), flush=True)


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
    peak, _, peak_src = measured_peaks()
    alg = n_pos * (4 * 20 * 4 + 4) + 3 * n_pos * 8          # lists in, alpha out; three selection passes over (alpha, position)
    print(json.dumps({"metric": "acceptance-rate positions/s", "value": n_pos / (ms * 1e-3), "unit": "positions/s", "ms_per_call": ms,
                      "steps": args.steps, "config": {"workload": "acceptance", "n_pos": n_pos, "top_n": 20, "n_bins": n_bins, "bin_tokens": 2048},
                      "roofline": {"bound": "hbm", "achieved": alg / (ms * 1e-3) / 1e9, "peak": peak, "unit": "GB/s",
                                   "frac": alg / (ms * 1e-3) / 1e9 / peak, "peak_source": peak_src, "algorithmic_bytes_per_call": alg},
                      "bin_count": bc.cpu().tolist(), "bin_5pct": [round(float(x), 4) for x in bq.cpu().tolist()]}), flush=True)


def relaunch_under_torchrun(args) -> int:
    """`--gpus N` without a torchrun environment: start the N replica processes here (one per GPU, rendezvous on
    127.0.0.1) and hand their output through."""
    port = 29600 + os.getpid() % 300
    cmd = [sys.executable, "-m", "torch.distributed.run", "--nnodes=1", f"--nproc-per-node={args.gpus}", "--master-addr", "127.0.0.1",
           "--master-port", str(port), os.path.abspath(__file__)] + sys.argv[1:]
    return subprocess.call(cmd)


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=20)
    ap.add_argument("--warmup", type=int, default=5)
    ap.add_argument("--workload", default="cfg4", choices=[c for c in W.CONFIGS if c not in ("cfg1", "cfg1_dense")],
                    help="cfg4 (default): the 36-layer step, the largest single-GPU configuration, with the single-layer configs in per_config")
    ap.add_argument("--pools", type=int, default=4, help="cfg4 only: distinct K/V pools the 36 layers rotate over (~14 GiB each)")
    ap.add_argument("--impl", default="sparrow", choices=["sparrow", "reference"])
    ap.add_argument("--no-per-config", action="store_true", help="cfg4 only: skip the per_config block (cfg2, cfg3, cfg5 single-layer results)")
    ap.add_argument("--rollout", type=int, default=0, metavar="T", help="time a T-step sparse rollout against the dense rollout (SURVEY 8(f)-1)")
    ap.add_argument("--rollout-bucket", type=int, default=512, help="steps per CUDA graph / per row of the rollout table")
    ap.add_argument("--table4", action="store_true", help="page-size sweep at budget 1024 (PAPER.md Table 4) instead of the step benchmark")
    ap.add_argument("--acceptance", action="store_true", help="time sparrow_acceptance (SURVEY 8(f)-3) instead of the step benchmark")
    ap.add_argument("--landmark", default="minmax", choices=["minmax", "mean"],
                    help="page landmark: per-channel min/max (north_star's default, 512 B) or the mean key (the paper's cost model, 256 B)")
    ap.add_argument("--kv-layout", default="hnd", choices=["hnd", "nhd"],
                    help="single-layer configs: K/V pools packed [page][kv-head][token][128] (default) or [page][token][kv-head][128] through the stride fields")
    ap.add_argument("--deterministic", action="store_true",
                    help="run the decode with SPARROW_FLAG_DETERMINISTIC (fixed tile hand-out: bit-reproducible out / lse)")
    ap.add_argument("--launch-check", action="store_true", help="only bring up the N ranks, barrier, and print their count (CPU: gloo)")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-check", action="store_true", help="skip the oracle self-check before timing")
    args = ap.parse_args()
    args.warmup = max(args.warmup, 3)
    if args.landmark == "mean":
        args.no_cpu_baseline = True      # the timed CPU baseline is the default (min/max) path's oracle

    if args.gpus > 1 and "WORLD_SIZE" not in os.environ:
        sys.exit(relaunch_under_torchrun(args))
    rank, local_rank, world = D.env_world()
    if args.launch_check:
        D.init("nccl" if torch.cuda.is_available() else "gloo")
        if torch.cuda.is_available():
            torch.cuda.set_device(local_rank)
        D.barrier()
        n = D.sum_over_ranks(1.0, device=f"cuda:{local_rank}" if torch.cuda.is_available() else "cpu")
        if rank == 0:
            print(json.dumps({"launch_check": True, "n_gpus": int(n), "world_size": world, "requested": args.gpus}), flush=True)
        D.barrier()
        return
    if args.impl == "reference":
        run_reference(args, rank)
        return
    assert torch.cuda.is_available(), "bench.py needs a CUDA device: there is no CPU fallback"
    torch.cuda.set_device(local_rank)
    dev = torch.device("cuda", local_rank)
    D.init("nccl")
    if args.rollout:
        return run_rollout(args, rank, dev)
    if args.table4:
        return run_table4(args, rank, dev)
    if args.acceptance:
        return run_acceptance(args, rank, dev)
    if args.workload != "cfg4":
        line = run_single(args, args.workload, rank, local_rank, world, dev)
    else:
        line = run_cfg4(args, rank, local_rank, world, dev)
        if not args.no_per_config and args.landmark == "minmax":
            per = {}
            for cfg in ("cfg2", "cfg3", "cfg5"):
                r = run_single(args, cfg, rank, local_rank, world, dev, headline=False)
                if rank == 0:
                    per[cfg] = {k: r[k] for k in ("value", "ms_per_step", "config", "roofline", "kernels", "sparse_path_GBs", "sparse_path_frac",
                                                  "speedup_vs_dense", "ideal_speedup_bytes_ratio", "cost_model", "e2e", "self_check", "cpu_baseline")
                                if k in r}
            if rank == 0:
                line["per_config"] = per
    if rank == 0:
        print(json.dumps(line), flush=True)


if __name__ == "__main__":
    main()
