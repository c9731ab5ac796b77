"""Seeded synthetic workloads shaped like the paper's Qwen3 rollouts (BASELINE.json configs 1-5).

This module serves BOTH the CUDA path and the CPU oracle and therefore holds none of the method's
arithmetic: it draws lengths, page tables, q, K and V, plants pages (reading R19) and
describes the schedule as plain data.  B(L), forced pages, scores, top-k and attention are each
written twice elsewhere (oracle/ and csrc/), never here.

The paper measures on AIME24 prompts x8 with a 32K cutoff and Polaris rollouts;
those items and the Qwen3 weights are not available, so these inputs take only their *shapes*
(Qwen3 GQA head counts, page 16, contexts up to ~40K tokens) and stand in for them.
"""
from __future__ import annotations

import math
from dataclasses import dataclass, field
from typing import Dict, List, Optional

import numpy as np
import torch

PAGE = 16
HEAD_DIM = 128


def _sched(kind, S, W, **kw) -> dict:
    d = dict(kind=kind, sink_tokens=S, local_tokens=W, fixed_tokens=0, floor_tokens=0,
             f0_ppm=0, f1_ppm=0, L0=0, L1=1, table_pages=(), bin_tokens=2048)
    d.update(kw)
    return d


# Plain-data descriptions of BASELINE.json's configs.
CONFIGS: Dict[str, dict] = {
    "cfg1": dict(n_seq=2, Hq=4, Hkv=2, lengths=("list", [1024, 1500]), plant=False,
                 schedule=_sched("fixed", 16, 64, fixed_tokens=256)),
    "cfg1_dense": dict(n_seq=2, Hq=4, Hkv=2, lengths=("list", [1024, 1500]), plant=False,
                       schedule=_sched("fixed", 16, 64, fixed_tokens=4096)),
    "cfg2": dict(n_seq=64, Hq=16, Hkv=8, lengths=("uniform", 4096, 16384), plant=True,
                 schedule=_sched("clamp_frac", 64, 512, f0_ppm=125000, floor_tokens=2048)),
    "cfg3": dict(n_seq=128, Hq=32, Hkv=8, lengths=("uniform", 8192, 32768), plant=True,
                 schedule=_sched("linear_frac", 64, 512, f0_ppm=250000, f1_ppm=62500, L0=8192, L1=32768,
                                 floor_tokens=2048)),
    # one layer pool of config 4 (36 layers = 36 calls over rotating pools, layers 0-1 dense)
    "cfg4": dict(n_seq=256, Hq=32, Hkv=8, lengths=("lognormal", 12288, 0.7, 1024, 32768), plant=True,
                 schedule=_sched("linear_frac", 64, 512, f0_ppm=250000, f1_ppm=62500, L0=8192, L1=32768,
                                 floor_tokens=2048), n_layers=36, dense_layers=2),
    "cfg5": dict(n_seq=32, Hq=40, Hkv=8, lengths=("uniform", 24576, 40960), plant=True,
                 schedule=_sched("clamp_frac", 64, 512, f0_ppm=50000, floor_tokens=1024)),
}


@dataclass
class Workload:
    name: str
    n_seq: int
    Hq: int
    Hkv: int
    schedule: dict
    seq_lens: torch.Tensor        # int32 [n]            (device)
    page_table: torch.Tensor      # int32 [n][max_pages] (device), logical -> physical, padding = 0
    q: torch.Tensor               # bf16  [n][Hq][128]
    k_cache: torch.Tensor         # bf16  [n_phys][Hkv][16][128]
    v_cache: torch.Tensor         # bf16  [n_phys][Hkv][16][128]
    sm_scale: float
    planted: Optional[List[List[np.ndarray]]] = None   # [seq][kv-head] -> planted logical pages
    seed: int = 0
    meta: dict = field(default_factory=dict)
    page_size: int = PAGE         # tokens per page: 16 (the paper's choice) or 32 / 64 / 128 (Table 4)

    @property
    def max_pages(self) -> int:
        return int(self.page_table.shape[1])

    @property
    def n_phys(self) -> int:
        return int(self.k_cache.shape[0])

    def host(self) -> dict:
        """Exact bit patterns as numpy (bf16 -> uint16) for the oracle."""
        def bits(t):
            return t.detach().contiguous().view(torch.int16).cpu().numpy().view(np.uint16)
        return dict(q=bits(self.q), k_cache=bits(self.k_cache), v_cache=bits(self.v_cache),
                    page_table=self.page_table.cpu().numpy().astype(np.int32),
                    seq_lens=self.seq_lens.cpu().numpy().astype(np.int32))


def host_subset(wl: "Workload", idx) -> dict:
    """Host view (exact bit patterns, as Workload.host) of the sequences `idx` only, with the K/V pools COMPACTED to
    the pages those sequences own and the page table renumbered accordingly -- data movement only, so that a checker
    can look at a few sequences of a 13 GiB pool without copying the pool.  Extra keys: 'seq_index' (the original
    sequence numbers, in row order) and 'phys_ids' (original physical page of every compacted page)."""
    idx = [int(i) for i in idx]
    P = wl.page_size
    lens = wl.seq_lens.cpu()[idx].tolist()
    npg = [-(-L // P) for L in lens]
    pt_dev = wl.page_table[torch.as_tensor(idx, device=wl.page_table.device)]
    ids = torch.cat([pt_dev[j, :n] for j, n in enumerate(npg)]).long()
    new_pt = np.zeros((len(idx), max(npg)), dtype=np.int32)
    o = 0
    for j, n in enumerate(npg):
        new_pt[j, :n] = np.arange(o, o + n, dtype=np.int32)
        o += n

    def bits(t):
        return t.detach().contiguous().view(torch.int16).cpu().numpy().view(np.uint16)
    return dict(q=bits(wl.q[torch.as_tensor(idx, device=wl.q.device)]), k_cache=bits(wl.k_cache[ids]), v_cache=bits(wl.v_cache[ids]),
                page_table=new_pt, seq_lens=np.asarray(lens, dtype=np.int32), seq_index=np.asarray(idx, dtype=np.int64),
                phys_ids=ids.cpu().numpy())


def draw_lengths(spec, n_seq: int, gen: torch.Generator) -> List[int]:
    kind = spec[0]
    if kind == "list":
        assert len(spec[1]) == n_seq
        return [int(x) for x in spec[1]]
    if kind == "uniform":
        lo, hi = spec[1], spec[2]
        return torch.randint(lo, hi + 1, (n_seq,), generator=gen).tolist()
    if kind == "lognormal":           # R20: median, sigma in ln-space, rejection-sampled into [lo, hi]
        med, sig, lo, hi = spec[1:]
        out: List[int] = []
        while len(out) < n_seq:
            x = med * torch.exp(sig * torch.randn(4 * n_seq, generator=gen, dtype=torch.float64))
            out.extend(int(v) for v in x.tolist() if lo <= v <= hi)
        return out[:n_seq]
    raise ValueError(kind)


def make_workload(name: str = "custom", *, n_seq: int, Hq: int, Hkv: int, lengths, schedule: dict,
                  plant: bool = False, seed: int = 0, device="cpu", spare_pages: int = 3,
                  poison_tail=False, plant_scale: float = 3.0, plant_frac: float = 0.05,
                  chunk_pages: int = 8192, reserve_tokens: int = 0, page_size: int = PAGE, **_ignored) -> Workload:
    """Draw one batch.  Lengths, page tables and planted pages come from a CPU generator (so they do
    not depend on the device); q/K/V values come from a generator on ``device``."""
    dev = torch.device(device)
    cg = torch.Generator(device="cpu").manual_seed(seed)
    dg = torch.Generator(device=dev).manual_seed(seed + 7919)
    D, P = HEAD_DIM, page_size
    chunk_pages = max(1, chunk_pages * PAGE // P)
    r = Hq // Hkv
    assert Hq == r * Hkv

    lens = draw_lengths(lengths, n_seq, cg)
    # pages each sequence owns: its cached tokens plus room for `reserve_tokens` more (the rollout loop appends into them)
    n_pages = [-(-(L + reserve_tokens) // P) for L in lens]
    max_pages = max(n_pages)
    n_phys = sum(n_pages) + spare_pages
    perm = torch.randperm(n_phys, generator=cg)          # scattered physical placement
    page_table = torch.zeros((n_seq, max_pages), dtype=torch.int32)
    owner = torch.full((n_phys,), -1, dtype=torch.int64)
    o = 0
    for i, npg in enumerate(n_pages):
        ids = perm[o:o + npg]
        page_table[i, :npg] = ids.to(torch.int32)
        owner[ids] = i
        o += npg

    q = torch.randn((n_seq, Hq, D), generator=dg, device=dev, dtype=torch.float32).to(torch.bfloat16)

    planted = None
    plant_mask = None
    if plant:
        planted = []
        plant_mask = torch.zeros((n_phys, Hkv), dtype=torch.bool)
        for i, npg in enumerate(n_pages):
            per_head = []
            n_pl = int(round(plant_frac * npg))
            for g in range(Hkv):
                lp = torch.randperm(npg, generator=cg)[:n_pl]
                plant_mask[page_table[i, lp].long(), g] = True
                per_head.append(np.sort(lp.numpy()))
            planted.append(per_head)
        # R19: offset = plant_scale * unit(sum of the group's query heads), added in fp32 before rounding
        gq = q.float().view(n_seq, Hkv, r, D).sum(2)
        U = plant_scale * gq / gq.norm(dim=-1, keepdim=True).clamp_min(1e-20)          # [n][Hkv][D]
        plant_mask = plant_mask.to(dev)
        owner_d = owner.to(dev)

    k_cache = torch.empty((n_phys, Hkv, P, D), dtype=torch.bfloat16, device=dev)
    v_cache = torch.empty((n_phys, Hkv, P, D), dtype=torch.bfloat16, device=dev)
    for a in range(0, n_phys, chunk_pages):
        b = min(a + chunk_pages, n_phys)
        kf = torch.randn((b - a, Hkv, P, D), generator=dg, device=dev, dtype=torch.float32)
        if plant:
            own = owner_d[a:b].clamp_min(0)
            off = U[own] * plant_mask[a:b].unsqueeze(-1)                                 # [c][Hkv][D]
            kf += off.unsqueeze(2)
        k_cache[a:b] = kf.to(torch.bfloat16)
        v_cache[a:b] = torch.randn((b - a, Hkv, P, D), generator=dg, device=dev, dtype=torch.float32).to(torch.bfloat16)

    if poison_tail:   # slots beyond the cached length must never influence any result
        for i, L in enumerate(lens):
            tail = L % P
            if tail:
                ph = int(page_table[i, L // P])
                if poison_tail == "nonfinite":      # what a torch.empty pool or a recycled page may hold
                    k_cache[ph, :, tail:, :] = float("nan")
                    v_cache[ph, :, tail:, :] = float("inf")
                else:
                    k_cache[ph, :, tail:, :] = 1.0e4
                    v_cache[ph, :, tail:, :] = -1.0e4

    return Workload(
        name=name, n_seq=n_seq, Hq=Hq, Hkv=Hkv, schedule=dict(schedule),
        seq_lens=torch.tensor(lens, dtype=torch.int32, device=dev),
        page_table=page_table.to(dev), q=q, k_cache=k_cache, v_cache=v_cache,
        sm_scale=1.0 / math.sqrt(D), planted=planted, seed=seed,
        meta=dict(lengths=lengths, n_pages_total=sum(n_pages), plant=plant), page_size=P,
    )


def make_config(name: str, *, seed: Optional[int] = None, device="cpu", **overrides) -> Workload:
    """One of BASELINE.json's configs ('cfg1', 'cfg1_dense', 'cfg2', ... 'cfg5')."""
    spec = dict(CONFIGS[name])
    spec.update(overrides)
    if seed is None:
        seed = 1000 * int("".join(ch for ch in name if ch.isdigit()) or 0)
    return make_workload(name, seed=seed, device=device, **spec)


def full_page_updates(wl: Workload):
    """(page_ids, n_valid) of every page the batch owns: the post-prefill bulk summarize call."""
    lens = wl.seq_lens.cpu().tolist()
    pt = wl.page_table.cpu()
    ids, nv = [], []
    for i, L in enumerate(lens):
        P = wl.page_size
        npg = -(-L // P)
        ids.append(pt[i, :npg])
        v = torch.full((npg,), P, dtype=torch.int32)
        if L % P:
            v[-1] = L % P
        nv.append(v)
    return torch.cat(ids).to(torch.int32), torch.cat(nv)


def just_filled_updates(wl: Workload):
    """(page_ids, n_valid) of pages that became full at this decode step (L % 16 == 0)."""
    lens = wl.seq_lens.cpu().tolist()
    pt = wl.page_table.cpu()
    P = wl.page_size
    ids = [int(pt[i, L // P - 1]) for i, L in enumerate(lens) if L % P == 0 and L > 0]
    return torch.tensor(ids, dtype=torch.int32), torch.full((len(ids),), P, dtype=torch.int32)


def make_rollout_inputs(wl: Workload, n_steps: int, seed: int = 0):
    """Per-step inputs of a T-step rollout: q [T][n][Hq][128], k_new / v_new [T][n][Hkv][128],
    bf16 ~ N(0,1) from a seeded generator on the workload's device.  No method arithmetic here."""
    dev = wl.q.device
    g = torch.Generator(device=dev).manual_seed(seed + 104729)
    def draw(h):
        return torch.randn((n_steps, wl.n_seq, h, HEAD_DIM), generator=g, device=dev, dtype=torch.float32).to(torch.bfloat16)
    return draw(wl.Hq), draw(wl.Hkv), draw(wl.Hkv)


def make_acceptance_inputs(n_traj: int, max_len: int, top_n: int = 20, vocab: int = 2048, seed: int = 0, device="cpu"):
    """Synthetic stand-in for what the inference engine returns for the paper's divergence study: per
    generated token the top-N token ids and log-probabilities under the dense policy P and the sparse policy Q.
    Logits P ~ N(0, 2^2); Q = P + noise whose scale grows with the token position (the mismatch grows with length,
    PAPER.md:99-103).  Trajectory lengths uniform in [max_len / 4, max_len].  Input generation only."""
    dev = torch.device(device)
    cg = torch.Generator(device="cpu").manual_seed(seed)
    dg = torch.Generator(device=dev).manual_seed(seed + 15485863)
    lens = torch.randint(max(1, max_len // 4), max_len + 1, (n_traj,), generator=cg)
    positions = torch.cat([torch.arange(int(L), dtype=torch.int32) for L in lens]).to(dev)
    n_pos = int(positions.numel())
    out = {k: [] for k in ("ids_p", "logp_p", "ids_q", "logp_q")}
    for a in range(0, n_pos, 16384):
        pos = positions[a:a + 16384].float()
        lp = 2.0 * torch.randn((len(pos), vocab), generator=dg, device=dev)
        lq = lp + (0.05 + 0.6 * pos / max_len).unsqueeze(1) * torch.randn((len(pos), vocab), generator=dg, device=dev)
        for name, logits in (("p", lp), ("q", lq)):
            lsm = torch.log_softmax(logits, dim=-1)
            val, idx = lsm.topk(top_n, dim=-1)
            out["ids_" + name].append(idx.to(torch.int32)); out["logp_" + name].append(val.float())
    return {k: torch.cat(v).contiguous() for k, v in out.items()} | {"positions": positions, "lens": lens}
