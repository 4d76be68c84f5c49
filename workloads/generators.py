"""Seeded synthetic inputs for the ART decode-attention path.

This module serves BOTH the CPU oracle (tests) and the CUDA path (tests, bench): it
produces one payload that is handed to both.  It holds none of the method's
arithmetic: no softmax, no streaming update, no criterion, no traversal order.  The
only attention-flavoured thing here is the BASE POLICY that ART composes with
(PAPER.md:167-173): the block-score / top-k selection that decides which blocks are
eligible and in what priority, which the paper treats as an input to ART.

Stand-in statement: the paper measures on LongBench / RULER-NIAH with real model
weights.  None of that is available; these generators take the
paper's shapes (Mistral-7B / Llama-3.1-70B GQA geometry, contexts 2K-128K, batch
1-128, sink = 4 tokens per PAPER.md:483) and BASELINE.json's value distributions.
No benchmark item is reproduced.

All tensors are torch tensors on `device`; values are drawn in fp32 with a seeded
torch.Generator on that device, then rounded RNE to the KV dtype.  CPU and CUDA
draws differ bit-wise (different Philox streams); within one run the oracle and the
kernel always see the identical payload.
"""
from __future__ import annotations

from dataclasses import dataclass, field, replace
import math

import torch

BLOCK_TOKENS = 64
POLICY_DENSE, POLICY_SINK_WINDOW, POLICY_LIST = 0, 1, 2
LAYOUT_HND, LAYOUT_NHD = 0, 1
SEED_BASE = 260600024


@dataclass
class Workload:
    name: str
    batch: int
    num_q_heads: int
    num_kv_heads: int
    head_dim: int
    dtype: torch.dtype                 # torch.float32 or torch.bfloat16 (q, k, v share it)
    policy: int
    layout: int
    q: torch.Tensor                    # [B, Hq, d]
    k_cache: torch.Tensor              # HND: [pages, Hkv, 64, d]; NHD: [pages, 64, Hkv, d]
    v_cache: torch.Tensor
    block_table: torch.Tensor          # [B, max_blocks] int32, logical block -> physical page
    seq_lens: torch.Tensor             # [B] int32
    sink_tokens: int = 0
    window_tokens: int = 0
    eligible_blocks: torch.Tensor | None = None   # [B, Hkv, max_eligible] int32 (LIST)
    eligible_counts: torch.Tensor | None = None   # [B, Hkv] int32 (LIST)
    tau: float = 1e-5
    phi: float = 1e-3
    patience: int = 5
    probe_dim: int = 32
    notes: dict = field(default_factory=dict)

    @property
    def group_size(self) -> int:
        return self.num_q_heads // self.num_kv_heads

    def to(self, device) -> "Workload":
        mv = lambda t: None if t is None else t.to(device)
        return replace(self, q=mv(self.q), k_cache=mv(self.k_cache), v_cache=mv(self.v_cache),
                       block_table=mv(self.block_table), seq_lens=mv(self.seq_lens),
                       eligible_blocks=mv(self.eligible_blocks), eligible_counts=mv(self.eligible_counts))


# --------------------------------------------------------------------------- helpers

def _gen(seed: int, device) -> torch.Generator:
    g = torch.Generator(device=device)
    g.manual_seed(int(seed))
    return g


def _unit(x: torch.Tensor) -> torch.Tensor:
    return x / x.norm(dim=-1, keepdim=True).clamp_min(1e-30)


def _alloc_pages(seq_lens: torch.Tensor, gen: torch.Generator, device):
    """Random page permutation: block_table[b, blk] = physical page (every page used once)."""
    nblk = (seq_lens.to(torch.int64) + BLOCK_TOKENS - 1) // BLOCK_TOKENS
    total = int(nblk.sum())
    perm = torch.randperm(total, generator=gen, device=device).to(torch.int32)
    max_blocks = int(nblk.max()) if total > 0 else 1
    table = torch.zeros((len(seq_lens), max(max_blocks, 1)), dtype=torch.int32, device=device)
    off = 0
    for b, n in enumerate(nblk.tolist()):
        table[b, :n] = perm[off:off + n]
        off += n
    return table, total


def _store_sequence(cache: torch.Tensor, layout: int, pages: torch.Tensor, x_logical: torch.Tensor):
    """x_logical [nb, Hkv, 64, d] (logical block order) -> paged cache, rounded to its dtype."""
    x = x_logical.to(cache.dtype)
    if layout == LAYOUT_NHD:
        x = x.permute(0, 2, 1, 3)
    cache[pages.long()] = x


def _block_scores(q_b: torch.Tensor, k_b: torch.Tensor, L: int, G: int) -> torch.Tensor:
    """Base-policy block priority (SnapKV-like stand-in): mean over the
    group's G heads and the block's valid tokens of q_h . k_j.  q_b [Hq, d] fp32,
    k_b [nb, Hkv, 64, d] fp32 (already rounded to the KV dtype).  -> [Hkv, nb]."""
    nb, Hkv, n, d = k_b.shape
    qg = q_b.view(Hkv, G, d).sum(dim=1)                       # sum over heads of the group
    tok = torch.arange(nb * n, device=k_b.device).view(nb, n)
    valid = (tok < L).to(k_b.dtype)                           # [nb, 64]
    s = torch.einsum("gd,bgnd->gbn", qg, k_b) * valid[None]   # [Hkv, nb, 64]
    return s.sum(dim=-1) / (G * valid.sum(dim=-1).clamp_min(1.0))[None]


def _topk_lists(scores: torch.Tensor, k: int):
    """Descending score, ties -> lower block index first (reading R10).  scores [Hkv, nb]."""
    Hkv, nb = scores.shape
    k = min(k, nb)
    order = torch.argsort(scores, dim=-1, descending=True, stable=True)   # stable => lower index first on ties
    return order[:, :k].to(torch.int32), k


# --------------------------------------------------------------------------- generic builder

def make_workload(name: str, *, seed: int, batch: int, num_q_heads: int, num_kv_heads: int,
                  head_dim: int, seq_lens, dtype=torch.bfloat16, policy: int = POLICY_DENSE,
                  layout: int = LAYOUT_HND, device="cpu", q_scale: float = 1.0,
                  planted_frac: float = 0.0, planted_strength: float = 3.0, sink_plant: int = 0,
                  sink_tokens: int = 0, window_tokens: int = 0, topk_blocks: int = 0,
                  topk_frac: float = 0.0, recency_decay: tuple[float, float] | None = None,
                  needle: bool = False, heavy_keys: tuple[int, float] | None = None,
                  poison_tail: bool = True, tau: float = 1e-5, phi: float = 1e-3,
                  patience: int = 5, probe_dim: int = 32) -> Workload:
    """Build one synthetic decode step.

    K, V ~ N(0,1); Q ~ N(0,1) * q_scale.
    planted_frac/planted_strength/sink_plant: config-1 recipe (query-aligned keys, sinks).
    topk_blocks / topk_frac: LIST policy from block scores.
    recency_decay=(lo, hi): variant R, key -= lambda * age * sum_h q_hat_h, lambda log-uniform.
    needle: config-4 recipe.  heavy_keys=(count_per_end, strength): config-0 recipe.
    poison_tail: slots of the last page beyond seq_len are filled with NaN (must be masked).
    """
    dev = torch.device(device)
    gen = _gen(seed, dev)
    B, Hq, Hkv, d = batch, num_q_heads, num_kv_heads, head_dim
    G = Hq // Hkv
    seq_lens_t = torch.as_tensor(seq_lens, dtype=torch.int32, device=dev).reshape(B)
    block_table, total_pages = _alloc_pages(seq_lens_t, gen, dev)
    shape = (max(total_pages, 1), Hkv, BLOCK_TOKENS, d) if layout == LAYOUT_HND else \
            (max(total_pages, 1), BLOCK_TOKENS, Hkv, d)
    k_cache = torch.zeros(shape, dtype=dtype, device=dev)
    v_cache = torch.zeros(shape, dtype=dtype, device=dev)

    q32 = torch.randn((B, Hq, d), generator=gen, device=dev, dtype=torch.float32) * q_scale
    q = q32.to(dtype)
    qf = q.to(torch.float32)                                  # what the kernels really see
    qhat = _unit(qf)                                          # [B, Hq, d]
    qhat_group_sum = qhat.view(B, Hkv, G, d).sum(dim=2)       # [B, Hkv, d]

    notes: dict = {}
    max_elig = 0
    lists, counts = [], []
    want_list = policy == POLICY_LIST
    if recency_decay is not None:
        lo, hi = recency_decay
        u = torch.rand((B, Hkv), generator=gen, device=dev)
        lam = torch.exp(math.log(lo) + u * (math.log(hi) - math.log(lo)))
        notes["recency_lambda"] = lam.cpu()
    if needle:
        notes["needle_block"] = []

    for b in range(B):
        L = int(seq_lens_t[b])
        nb = (L + BLOCK_TOKENS - 1) // BLOCK_TOKENS
        if nb == 0:
            if want_list:
                lists.append(torch.zeros((Hkv, 0), dtype=torch.int32, device=dev)); counts.append(0)
            continue
        kb = torch.randn((nb, Hkv, BLOCK_TOKENS, d), generator=gen, device=dev, dtype=torch.float32)
        vb = torch.randn((nb, Hkv, BLOCK_TOKENS, d), generator=gen, device=dev, dtype=torch.float32)
        kflat = kb.permute(1, 0, 2, 3).reshape(Hkv, nb * BLOCK_TOKENS, d)   # view: [Hkv, tokens, d]
        vflat = vb.permute(1, 0, 2, 3).reshape(Hkv, nb * BLOCK_TOKENS, d)
        # NOTE: permute+reshape copies; write results back below
        if planted_frac > 0.0:
            npl = int(round(planted_frac * L))
            for g in range(Hkv):
                pos = torch.randperm(L, generator=gen, device=dev)[:npl]
                heads = g * G + (torch.arange(npl, device=dev) % G)
                kflat[g, pos] += planted_strength * qhat[b, heads]
        if sink_plant > 0:
            ns = min(sink_plant, L)
            kflat[:, :ns] += planted_strength * qhat_group_sum[b][:, None, :]
        if heavy_keys is not None:
            cnt, strength = heavy_keys
            last_blk_start = (nb - 1) * BLOCK_TOKENS
            positions = list(range(cnt)) + list(range(last_blk_start, last_blk_start + cnt))
            for i, p in enumerate(positions):
                for g in range(Hkv):
                    kflat[g, p] = strength * qhat[b, g * G + (i % G)]
        if needle:
            nblk = int(torch.randint(0, nb, (1,), generator=gen, device=dev))
            notes["needle_block"].append(nblk)
            tok = torch.arange(BLOCK_TOKENS, device=dev)
            for g in range(Hkv):
                heads = g * G + (tok % G)
                kflat[g, nblk * BLOCK_TOKENS:(nblk + 1) * BLOCK_TOKENS] = 5.0 * qhat[b, heads]
                r = _unit(torch.randn((d,), generator=gen, device=dev))
                vflat[g, nblk * BLOCK_TOKENS:(nblk + 1) * BLOCK_TOKENS] = 10.0 * r
        if recency_decay is not None:
            age = (nb - 1) - (torch.arange(nb * BLOCK_TOKENS, device=dev) // BLOCK_TOKENS)   # blocks behind newest
            kflat -= lam[b][:, None, None] * age[None, :, None].float() * qhat_group_sum[b][:, None, :]
        kb = kflat.view(Hkv, nb, BLOCK_TOKENS, d).permute(1, 0, 2, 3)
        vb = vflat.view(Hkv, nb, BLOCK_TOKENS, d).permute(1, 0, 2, 3)
        kb_r = kb.to(dtype)                                   # RNE to the KV dtype
        if want_list:
            sc = _block_scores(qf[b], kb_r.to(torch.float32), L, G)
            kk = topk_blocks if topk_blocks > 0 else max(1, int(round(topk_frac * nb)))
            lst, kk = _topk_lists(sc, kk)
            lists.append(lst); counts.append(kk); max_elig = max(max_elig, kk)
        if poison_tail and L % BLOCK_TOKENS != 0:
            kb_r = kb_r.clone(); vb = vb.clone()
            kb_r[nb - 1, :, L % BLOCK_TOKENS:] = float("nan")
            vb[nb - 1, :, L % BLOCK_TOKENS:] = float("nan")
        pages = block_table[b, :nb]
        _store_sequence(k_cache, layout, pages, kb_r)
        _store_sequence(v_cache, layout, pages, vb)
        del kb, vb, kflat, vflat, kb_r

    eligible_blocks = eligible_counts = None
    if want_list:
        max_elig = max(max_elig, 1)
        eligible_blocks = torch.zeros((B, Hkv, max_elig), dtype=torch.int32, device=dev)
        eligible_counts = torch.zeros((B, Hkv), dtype=torch.int32, device=dev)
        for b in range(B):
            kk = counts[b]
            if kk > 0:
                eligible_blocks[b, :, :kk] = lists[b]
            eligible_counts[b, :] = kk

    return Workload(name=name, batch=B, num_q_heads=Hq, num_kv_heads=Hkv, head_dim=d, dtype=dtype,
                    policy=policy, layout=layout, q=q, k_cache=k_cache, v_cache=v_cache,
                    block_table=block_table, seq_lens=seq_lens_t, sink_tokens=sink_tokens,
                    window_tokens=window_tokens, eligible_blocks=eligible_blocks,
                    eligible_counts=eligible_counts, tau=tau, phi=phi, patience=patience,
                    probe_dim=probe_dim, notes=notes)


# --------------------------------------------------------------------------- BASELINE.json configs

def _uniform_lens(seed: int, batch: int, lo: int, hi: int):
    g = torch.Generator(device="cpu"); g.manual_seed(seed + 7)
    return torch.randint(lo, hi + 1, (batch,), generator=g, dtype=torch.int64).to(torch.int32)


def config(index: int, *, device="cpu", variant: str = "", scale: float = 1.0, batch: int | None = None,
           sub: str = "a", layout: int = LAYOUT_HND, **over) -> Workload:
    """BASELINE.json `configs[index]` as a concrete generator.

    variant "" = literal; "R" = recency-decay supplement (configs 1-4); "c" = config 0 with
    heavy-key strength 200.  `scale` shrinks the context (tests); `batch` overrides B.
    Config 3 has two policies: sub="a" sink(4)+window(4096), sub="b" top-k(64 blocks).
    """
    seed = SEED_BASE + 1000 * index
    rd = (0.01, 0.3) if variant == "R" else None
    sc = lambda n: max(BLOCK_TOKENS, int(n * scale) // BLOCK_TOKENS * BLOCK_TOKENS)
    if index == 0:
        strength = 200.0 if variant == "c" else 4.0
        kw = dict(seed=seed, batch=batch or 1, num_q_heads=4, num_kv_heads=1, head_dim=64,
                  seq_lens=[sc(2048)] * (batch or 1), dtype=torch.float32, policy=POLICY_DENSE,
                  q_scale=1.0 / 8.0, heavy_keys=(8, strength))
        name = "cfg0_tiny_fp32" + ("_c" if variant == "c" else "")
    elif index == 1:
        B = batch or 8
        kw = dict(seed=seed, batch=B, num_q_heads=32, num_kv_heads=8, head_dim=128,
                  seq_lens=[sc(32768)] * B, policy=POLICY_DENSE, planted_frac=0.01, sink_plant=4,
                  recency_decay=rd)
        name = "cfg1_mistral7b_dense" + ("_R" if rd else "")
    elif index == 2:
        B = batch or 16
        kw = dict(seed=seed, batch=B, num_q_heads=64, num_kv_heads=8, head_dim=128,
                  seq_lens=[sc(65536)] * B, policy=POLICY_LIST, planted_frac=0.01, sink_plant=4,
                  topk_frac=0.25, recency_decay=rd)
        name = "cfg2_llama70b_top25" + ("_R" if rd else "")
    elif index == 3:
        B = batch or 128
        lens = _uniform_lens(seed, B, max(BLOCK_TOKENS, int(4096 * scale)), max(BLOCK_TOKENS, int(32768 * scale)))
        kw = dict(seed=seed, batch=B, num_q_heads=32, num_kv_heads=8, head_dim=128, seq_lens=lens,
                  planted_frac=0.01, sink_plant=4, recency_decay=rd)
        if sub == "a":
            kw.update(policy=POLICY_SINK_WINDOW, sink_tokens=4, window_tokens=max(BLOCK_TOKENS, int(4096 * scale)))
            name = "cfg3a_batch128_sink_window"
        else:
            kw.update(policy=POLICY_LIST, topk_blocks=max(1, int(64 * scale)))
            name = "cfg3b_batch128_top64"
        name += "_R" if rd else ""
    elif index == 4:
        B = batch or 4
        kw = dict(seed=seed, batch=B, num_q_heads=32, num_kv_heads=8, head_dim=128,
                  seq_lens=[sc(131072)] * B, policy=POLICY_DENSE, needle=True, recency_decay=rd)
        name = "cfg4_needle_128k" + ("_R" if rd else "")
    else:
        raise ValueError("config index 0..4")
    kw.update(over)
    return make_workload(name, device=device, layout=layout, **kw)


def with_query_tokens(w: Workload, m: int, *, seed: int, jitter: float = 0.5) -> Workload:
    """Multi-token variant of a decode step (speculative decode / the tail of a chunked prefill):
    q becomes [B, m, Hq, d].  The LAST query token is the workload's own; the m - 1 before it are that query plus
    N(0, jitter^2) noise per coordinate (scaled by the query's rms), as neighbouring positions of one sequence
    ask similar questions.  The cache is untouched: its last m positions are taken to be the query tokens'."""
    from dataclasses import replace
    gen = _gen(seed, w.q.device)
    q32 = w.q.to(torch.float32)
    rms = q32.pow(2).mean(dim=-1, keepdim=True).sqrt()
    toks = [q32 + jitter * rms * torch.randn(q32.shape, generator=gen, device=w.q.device, dtype=torch.float32)
            for _ in range(m - 1)] + [q32]
    return replace(w, q=torch.stack(toks, dim=1).to(w.dtype).contiguous())

